// dmat_long.cuh -- k_dmat_long, the distortion-matrix kernel for LONG forests (eqs. 2.6-2.7, PAPER.md:91-98;
// native-resolution shapes, PAPER.md:79, 140-145 and DESIGN.md NEXT-3): up to LYA_LONG_TILE pixels per forest,
// pixel spacing down to a sixteenth of the r_par bin width (LYA_DS_MAX_LONG).  Included by dmat.cu only.
//
// A forest pair of such forests holds 10^4..10^5 in-grid pixel pairs and hundreds of kept ones, so ONE CTA works
// on one forest pair (the fast kernels give a forest pair to one warp), every phase spread over its warps:
//  stage    both forests, (chi, ea) / eg and the stage-4 pixel keys, once for the CTA;
//  windows  threads over the rows of p (lya_row_window, exact), block-wide prefix sum of the window sizes;
//  pass A   tasks (16-row group, side of chi_i = chi_j), claimed by the warps; each warp walks its tasks with
//           dm_walk (dmat_fast.cuh: lanes own diagonals ds apart and hold their table entry in registers) into
//           a table of its OWN; the tables are then summed into table 0 and its non-zero entries listed;
//  bands    the rows are cut into bands of about DL_KCAP / 2 expected kept pairs; per band the balanced stage-4
//           scan over all threads queues the kept pairs, and the warps claim batches of DL_KBATCH of them for the
//           drain: T1, T2 over the row window, T3 over the rows whose window holds j (an interval around i), T4
//           with lanes over the non-zero entries of table 0 and four kept pairs per entry read.
// Every update is one red.global.add.f64 into Dn (transposed bin order), as in k_dmat_fast.
#pragma once
#include "dmat_fast.cuh"

namespace {

#ifndef LYA_DL_WARPS
#define LYA_DL_WARPS 14
#endif
constexpr int DL_T = LYA_LONG_TILE;
constexpr int DL_WARPS = LYA_DL_WARPS, DL_THREADS = DL_WARPS * 32;
constexpr int DL_TP = ((DL_T + 15) / 16) * 16 + 2;      // rows of p incl. sentinel rows (walks cover whole row groups)
constexpr int DL_TQ = DL_T + 2 * FD_PAD + 2;            // q incl. sentinels either side and the pad pixel of an odd forest
constexpr int DL_KCAP = 2048;                           // kept pairs queued per band
#ifndef LYA_DL_KBATCH
#define LYA_DL_KBATCH 8
#endif
constexpr int DL_KBATCH = LYA_DL_KBATCH;                // kept pairs a warp drains together
#ifndef LYA_DL_ROWS
#define LYA_DL_ROWS 16
#endif
constexpr int DL_ROWS = LYA_DL_ROWS;                    // rows of p per pass-A task (even, <= 32)
constexpr int DL_RPT = (DL_T + DL_THREADS - 1) / DL_THREADS;   // rows per thread in the prefix sum
static_assert(DL_T <= 0xffff && (DL_T & (DL_T - 1)) == 0 && DL_KBATCH <= 32 && DL_KCAP >= 2 * DL_T, "record layout, search steps, one row fits the queue twice");

struct DlDrainWarp {                                    // per warp: one batch of kept pairs
    double2 kc01[DL_KBATCH], kc23[DL_KBATCH];           // om (1, u_j), om (u_i, u_i u_j)
    unsigned rowoff[DL_KBATCH];                         // A * n_bins: the row of Dn
    unsigned short ilo[DL_KBATCH], ihi[DL_KBATCH];      // rows of p whose window holds j
};
struct __align__(16) DlShared {
    double2 pce[DL_TP], qce[DL_TQ];                     // (chi, ea); q has FD_PAD sentinels either side
    double peg[DL_TP], qeg[DL_TQ];                      // eg
    unsigned long long qk[DL_T], pk[DL_T];              // stage-4 keys of the pixels
    DlDrainWarp dw[DL_WARPS];
    unsigned pre[DL_T + 2];                             // pre[i] = in-window pairs of the rows before i
    unsigned short jlo[DL_T + 4], jx[DL_T + 4], jhi[DL_T + 4];   // exact windows (row len = stop row of the mask scan)
    unsigned kept[DL_KCAP];                             // (i << 16) | j
    unsigned short nz[FD_SLOTS + 2];                    // non-zero entries of table 0
    unsigned wsum[32];
    unsigned nkept, nnz, next_task, next_batch;
    long long cur;                                      // forest pair of the CTA
};
constexpr size_t DL_SHARED_BYTES = (sizeof(DlShared) + 15) & ~(size_t)15;
constexpr size_t DL_SMEM_BYTES = DL_SHARED_BYTES + sizeof(DmTable) * DL_WARPS;
static_assert(DL_SMEM_BYTES <= (size_t)FD_SMEM_MAX, "k_dmat_long shared memory");

// T2 / T3 of one kept pair over the pixels [lo, hi) of one forest (ce, eg) against the fixed pixel chi_fix of the
// other: Dn[row][bin] += m0 * ea + mx * eg, one pixel per lane.  (With fine pixels several lanes of an instruction
// reduce onto the same bin; adding such runs up first -- across lanes with shuffles, or with each lane on 3..8
// consecutive pixels -- was measured no faster or slower at every spacing: profiles/r2i_next3_long_forests.md.)
template <bool POW2>
__device__ __forceinline__ void dl_t23(const BinParams &bp, const PairBin &g, const double2 *ce, const double *eg, int lo, int hi,
                                       double chi_fix, double m0, double mx, double *row, int lane, unsigned &n_red)
{
#pragma unroll 1
    for (int t = lo + lane; t < hi; t += 32) {
        const double2 v = ce[t];
        dm_red(row + (unsigned)dm_bin_in<POW2>(bp, g, chi_fix, v.x), fma(mx, eg[t], m0 * v.y));
        n_red += 1u;
    }
}

// drain of n <= DL_KBATCH kept pairs (kept[e] = (i << 16) | j) by one warp: T1..T4
template <bool POW2>
__device__ __forceinline__ void dl_drain(DlShared &sh, DlDrainWarp &dw, const DmTable &tb, const unsigned *kept, int n, int mp,
                                         const DmFastParams &P, const PairBin &g, long long offp, long long offq,
                                         int c0, int nnz, int lane, unsigned &n_red)
{
    const BinParams &bp = P.bp;
    const unsigned nb = (unsigned)(bp.n_par * bp.n_perp);
    const double2 *qce = sh.qce + FD_PAD;
    const double *qeg = sh.qeg + FD_PAD;
    double *const Dn = P.Dn;
    if (lane < n) {
        const unsigned rec = kept[lane];
        const int i = (int)(rec >> 16), j = (int)(rec & 0xffffu);
        const unsigned A = (unsigned)dm_bin_in<POW2>(bp, g, sh.pce[i].x, qce[j].x);
        const double om = P.prep.w[offp + i] * P.prep.w[offq + j], ui = P.prep.u[offp + i], uj = P.prep.u[offq + j];
        const double omi = om * ui;
        dw.kc01[lane] = make_double2(om, om * uj);
        dw.kc23[lane] = make_double2(omi, omi * uj);
        dw.rowoff[lane] = A * nb;
        // rows of p whose window holds j: an interval around i (the in-grid region is a band in chi_i - chi_j cut by
        // a half-plane in chi_i + chi_j); fixed trip count
        int il = 0, ih = i + 1;
#pragma unroll
        for (int st = DL_T / 2; st; st >>= 1) {
            const int m = il + st, m2 = ih + st;
            if (m <= i) { const unsigned lo2 = sh.jlo[m - 1]; if (!((unsigned)j - lo2 < (unsigned)sh.jhi[m - 1] - lo2)) il = m; }
            if (m2 <= mp) { const unsigned lo2 = sh.jlo[m2 - 1]; if ((unsigned)j - lo2 < (unsigned)sh.jhi[m2 - 1] - lo2) ih = m2; }
        }
        dw.ilo[lane] = (unsigned short)il; dw.ihi[lane] = (unsigned short)ih;
        dm_red(Dn + (A * nb + A), om);                                                // T1
        dm_red(P.Wd + A, om);
        n_red += 2u;
    }
    __syncwarp();
#pragma unroll 1
    for (int e = 0; e < n; ++e) {
        const unsigned rec = kept[e];
        const int i = (int)(rec >> 16), j = (int)(rec & 0xffffu);
        const double2 c01 = dw.kc01[e];
        const double m0 = -c01.x, m1 = -c01.y, m2 = -dw.kc23[e].x;
        const double ci = sh.pce[i].x, cj = qce[j].x;
        const unsigned row = dw.rowoff[e];
        const int jh = sh.jhi[i], ih = dw.ihi[e];
        const int jl = sh.jlo[i], il = dw.ilo[e];
        dl_t23<POW2>(bp, g, qce, qeg, jl, jh, ci, m0, m1, Dn + row, lane, n_red);          // T2
        dl_t23<POW2>(bp, g, sh.pce, sh.peg, il, ih, cj, m0, m2, Dn + row, lane, n_red);    // T3
    }
    const unsigned col0 = (unsigned)(c0 * bp.n_par);
    for (int e0 = 0; e0 < n; e0 += FD_T4B) {                                          // T4
        double2 k01[FD_T4B], k23[FD_T4B];
        unsigned ro[FD_T4B];
#pragma unroll
        for (int k = 0; k < FD_T4B; ++k) {
            const int e = min(e0 + k, n - 1);
            k01[k] = dw.kc01[e]; k23[k] = dw.kc23[e];
            ro[k] = dw.rowoff[e] + col0;
        }
        const int m = min(FD_T4B, n - e0);
#pragma unroll 1
        for (int t = lane; t < nnz; t += 32) {
            const unsigned slot = sh.nz[t];
            const double2 a = tb.H01[slot], b = tb.H23[slot];
#pragma unroll
            for (int k = 0; k < FD_T4B; ++k)
                if (k < m) dm_red(Dn + (ro[k] + slot), fma(k23[k].y, b.y, fma(k23[k].x, b.x, fma(k01[k].y, a.y, k01[k].x * a.x))));
        }
        if (lane == 0) n_red += (unsigned)(m * nnz);
    }
    __syncwarp();
}

template <bool POW2, bool CHECK>
__global__ void __launch_bounds__(DL_THREADS, 1) k_dmat_long(DmFastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DlShared &sh = *(DlShared *)smem_raw;
    DmTable *tables = (DmTable *)(smem_raw + DL_SHARED_BYTES);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const BinParams bp = P.bp;
    const unsigned npar = (unsigned)bp.n_par;
    const int n_slots = bp.n_par * LYA_NCOL;                  // real slots; slot n_slots is the garbage entry
    for (int t = tid; t < DL_WARPS * FD_SLOTS; t += DL_THREADS) {
        tables[t / FD_SLOTS].H01[t % FD_SLOTS] = make_double2(0.0, 0.0);
        tables[t / FD_SLOTS].H23[t % FD_SLOTS] = make_double2(0.0, 0.0);
    }
    if (tid < FD_PAD) { sh.qce[tid] = make_double2(LYA_CHI_SENTINEL, 0.0); sh.qeg[tid] = 0.0; }
    const double2 *qce = sh.qce + FD_PAD;
    const bool keep_none = P.thr > 0xffffffffull;              // reject_fraction = 1
    const unsigned thr32 = (unsigned)P.thr;
    // in-window pairs per band: about DL_KCAP / 2 kept pairs expected, and never less than one full row
    unsigned band_pairs = 0xffffffffu;
    {
        const double keepf = 1.0 - (double)P.thr / 4294967296.0;
        if (!keep_none && keepf * 4.0e9 > (double)(DL_KCAP / 2)) band_pairs = max((unsigned)((double)(DL_KCAP / 2) / keepf), (unsigned)DL_T);
    }
    DmTable &tb_own = tables[wid];
    const unsigned h01 = (unsigned)__cvta_generic_to_shared(tb_own.H01);
    unsigned long long evaluated = 0, kept_total = 0, binned_total = 0, n_red = 0;
    unsigned conflicts = 0;
    for (;;) {
        __syncthreads();                                       // the previous forest pair is finished by every warp
        if (tid == 0) sh.cur = (long long)atomicAdd(&P.counters[4], 1ull);
        __syncthreads();
        const long long k = sh.cur;
        if (k >= P.n_pairs) break;
        const int2 e = ((const int2 *)P.pq)[k];
        const int p = e.x, q = e.y;
        const ForestHead hp = P.prep.head[p], hq = P.prep.head[q];
        const int mp = hp.len, mq = hq.len;
        if ((hp.flags | hq.flags) & 1) {
            if (tid == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_DEGENERATE);
            continue;
        }
        double s, c;
        lya_pair_sc(hp.ux, hp.uy, hp.uz, hq.ux, hq.uy, hq.uz, s, c);
        const PairBin g = lya_make_pairbin(bp, s, c);
        int c0;
        const int key = lya_pair_key<POW2>(bp, g, hp, hq, c0);
        if (key != LYA_KEY_LONG(bp.n_perp)) continue;         // cannot happen in the long range
        const unsigned lim = (unsigned)min(LYA_NCOL, bp.n_perp - c0);
        const int ds = lya_pair_stride(bp, g, hq);
        // ---- stage both forests and the stage-4 keys of their pixels ----
        {
            const double2 *sce = P.prep.ce + hp.off;
            const double2 *sg = (const double2 *)(P.prep.eg + hp.off);
            for (int t = tid; t < mp; t += DL_THREADS) sh.pce[t] = sce[t];
            for (int t = tid; 2 * t < mp; t += DL_THREADS) ((double2 *)sh.peg)[t] = sg[t];
            const double2 *tce = P.prep.ce + hq.off;
            const double2 *tg = (const double2 *)(P.prep.eg + hq.off);
            const int npad = (mq + 1) & ~1;
            for (int t = tid; t < npad; t += DL_THREADS) sh.qce[FD_PAD + t] = tce[t];      // (the pad pixel of an odd forest is a sentinel)
            for (int t = tid; 2 * t < npad; t += DL_THREADS) ((double2 *)(sh.qeg + FD_PAD))[t] = tg[t];
            if (tid < FD_PAD) { sh.qce[FD_PAD + npad + tid] = make_double2(LYA_CHI_SENTINEL, 0.0); sh.qeg[FD_PAD + npad + tid] = 0.0; }
            if (!keep_none) {
                for (int t = tid; t < mq; t += DL_THREADS) sh.qk[t] = lya_key_hi(P.seed, (unsigned long long)(hq.pix0 + t));
                for (int t = tid; t < mp; t += DL_THREADS) sh.pk[t] = lya_key_lo(P.seed, (unsigned long long)(hp.pix0 + t));
            }
        }
        __syncthreads();
        for (int t = mp + tid; t < ((mp + 15) & ~15) + 2; t += DL_THREADS) {            // sentinel rows (!= q's sentinel: r_par never 0)
            sh.pce[t] = make_double2(2.0 * LYA_CHI_SENTINEL, 0.0); sh.peg[t] = 0.0;
        }
        // ---- windows: threads over the rows of p ----
        const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;
        const double Tchi = (s > 0.0) ? (bp.rperp_max / s) * (1.0 + 1e-12) + 1e-9 : 1e300;
        for (int i = tid; i < mp; i += DL_THREADS) {
            int jlo, jx, jhi;
            lya_row_window_ilp<POW2, DL_T>(bp, g, qce, mq, sh.pce[i].x, R, Tchi, jlo, jx, jhi);
            sh.jlo[i] = (unsigned short)jlo; sh.jx[i] = (unsigned short)jx; sh.jhi[i] = (unsigned short)jhi;
            binned_total += (unsigned)(jhi - jlo);
        }
        if (tid == 0) { sh.jlo[mp] = 0; sh.jhi[mp] = 1; sh.next_task = 0u; }           // stop row: never empty, never left
        __syncthreads();
        {   // pre[i] = in-window pairs of the rows before i; pre[mp] = all of them
            const int r0 = DL_RPT * tid;
            unsigned wrow[DL_RPT], incl = 0;
#pragma unroll
            for (int kk = 0; kk < DL_RPT; ++kk) {
                wrow[kk] = (r0 + kk < mp) ? (unsigned)sh.jhi[r0 + kk] - sh.jlo[r0 + kk] : 0u;
                incl += wrow[kk];
            }
            const unsigned own = incl;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const unsigned v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
            if (lane == 31) sh.wsum[wid] = incl;
            __syncthreads();
            unsigned before = 0, total = 0;
            for (int w = 0; w < DL_WARPS; ++w) { const unsigned v = sh.wsum[w]; if (w < wid) before += v; total += v; }
            unsigned run = before + incl - own;
#pragma unroll
            for (int kk = 0; kk < DL_RPT; ++kk) {
                if (r0 + kk <= mp) sh.pre[r0 + kk] = run;
                run += wrow[kk];
            }
            if (tid == 0) sh.pre[mp] = total;
        }
        // ---- pass A: tasks (row group, side), each warp into its own table ----
        {
            const int n_tasks = 2 * ((mp + DL_ROWS - 1) / DL_ROWS);
            for (;;) {
                int task = 0;
                if (lane == 0) task = (int)atomicAdd(&sh.next_task, 1u);
                task = __shfl_sync(0xffffffffu, task, 0);
                if (task >= n_tasks) break;
                const int i0 = (task >> 1) * DL_ROWS, sgn = -(task & 1);
                const int i = i0 + lane;
                int lo = 1 << 20, hi = -(1 << 20), r0 = 1 << 20, r1 = -1;
                if (lane < DL_ROWS && i < mp) {
                    const int jl = sh.jlo[i], jh = sh.jhi[i], jx = sh.jx[i];
                    if (sgn == 0) { if (jx > jl) { lo = jl - i; hi = jx - 1 - i; r0 = i; r1 = i; } }
                    else if (jh > jx) { lo = jx - i; hi = jh - 1 - i; r0 = i; r1 = i; }
                }
                lo = __reduce_min_sync(0xffffffffu, lo); hi = __reduce_max_sync(0xffffffffu, hi);
                r0 = __reduce_min_sync(0xffffffffu, r0); r1 = __reduce_max_sync(0xffffffffu, r1);
                if (r1 >= r0)
                    dm_walk_any<POW2, CHECK>(sh, h01, r0 & ~1, r1 | 1, mq, lo, hi, ds, sgn, bp, g, (unsigned)c0, lim, npar, lane,
                                             evaluated, conflicts);
            }
        }
        __syncthreads();
        // ---- sum of the warps' tables into table 0 (the others are left all zero) ----
        for (int t = tid; t <= n_slots; t += DL_THREADS) {
            double2 a = tables[0].H01[t], b = tables[0].H23[t];
            for (int w = 1; w < DL_WARPS; ++w) {
                const double2 a2 = tables[w].H01[t], b2 = tables[w].H23[t];
                a.x += a2.x; a.y += a2.y; b.x += b2.x; b.y += b2.y;
                tables[w].H01[t] = make_double2(0.0, 0.0); tables[w].H23[t] = make_double2(0.0, 0.0);
            }
            if (t == n_slots) { a = make_double2(0.0, 0.0); b = a; }             // the garbage entry collects every out-of-grid product
            tables[0].H01[t] = a; tables[0].H23[t] = b;
        }
        __syncthreads();
        if (wid == 0) {                                        // non-zero entries of table 0
            int nnz = 0;
            for (int t0 = 0; t0 < n_slots; t0 += 32) {
                const int t = t0 + lane;
                bool nzf = false;
                if (t < n_slots) {
                    const double2 a = tables[0].H01[t], b = tables[0].H23[t];
                    nzf = (a.x != 0.0) | (a.y != 0.0) | (b.x != 0.0) | (b.y != 0.0);
                }
                const unsigned bal = __ballot_sync(0xffffffffu, nzf);
                if (nzf) sh.nz[nnz + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)t;
                nnz += __popc(bal);
            }
            if (lane == 0) sh.nnz = (unsigned)nnz;
        }
        __syncthreads();
        const int nnz = (int)sh.nnz;
        // ---- bands of rows: stage-4 scan over all threads, then the drain in batches claimed by the warps ----
        int ra = 0, rb = -1;
        while (ra < mp) {
            if (rb < 0) {                                      // last row end with at most band_pairs in-window pairs, at least one row
                const unsigned long long cap = (unsigned long long)sh.pre[ra] + band_pairs;
                int lo = ra + 1, hi = mp;
                while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if ((unsigned long long)sh.pre[mid] <= cap) lo = mid; else hi = mid - 1; }
                rb = lo;
            }
            if (tid == 0) { sh.nkept = 0u; sh.next_batch = 0u; }
            __syncthreads();
            if (!keep_none) {
                const unsigned base = sh.pre[ra], Mb = sh.pre[rb] - base;
                const unsigned K = (Mb + DL_THREADS - 1) / DL_THREADS;
                const unsigned first = base + min((unsigned)tid * K, Mb), last = base + min((unsigned)tid * K + K, Mb);
                int row = ra;                                  // last row with pre[row] <= first (fixed trip count)
#pragma unroll
                for (int st = DL_T / 2; st; st >>= 1) {
                    const int m = row + st;
                    if (m <= mp && sh.pre[m] <= first) row = m;
                }
                int j = (int)sh.jlo[row] + (int)(first - sh.pre[row]);
                int jend = (row >= mp) ? (1 << 30) : (int)sh.jhi[row];
                unsigned long long pki = sh.pk[min(row, DL_T - 1)];
                for (unsigned t = 0; t < K; ++t) {
                    if (j >= jend) {                           // next non-empty row (the stop row ends the search)
                        do { ++row; } while (sh.jlo[row] == sh.jhi[row]);
                        j = sh.jlo[row]; jend = (row >= mp) ? (1 << 30) : (int)sh.jhi[row];
                        pki = sh.pk[min(row, DL_T - 1)];
                    }
                    const unsigned h = lya_pair_hash32(pki, sh.qk[min(j, DL_T - 1)]);
                    if ((first + t < last) & (h >= thr32)) {
                        const unsigned idx = atomicAdd(&sh.nkept, 1u);
                        if (idx < DL_KCAP) sh.kept[idx] = ((unsigned)row << 16) | (unsigned)j;
                    }
                    ++j;
                }
            }
            __syncthreads();
            const unsigned nk = sh.nkept;
            if (nk > DL_KCAP) {                                // (32 sigma away at the band size chosen; halve the band and redo it)
                rb = ra + max(1, (rb - ra) >> 1);
                __syncthreads();
                continue;
            }
            if (tid == 0) kept_total += nk;
            unsigned n_red32 = 0;
            for (;;) {
                unsigned b = 0;
                if (lane == 0) b = atomicAdd(&sh.next_batch, 1u);
                b = __shfl_sync(0xffffffffu, b, 0);
                const unsigned e0 = b * DL_KBATCH;
                if (e0 >= nk) break;
                dl_drain<POW2>(sh, sh.dw[wid], tables[0], sh.kept + e0, (int)min((unsigned)DL_KBATCH, nk - e0), mp, P, g,
                               hp.off, hq.off, c0, nnz, lane, n_red32);
            }
            n_red += n_red32;
            ra = rb; rb = -1;
            __syncthreads();
        }
        // ---- table 0 back to all zero ----
        for (int t = tid; t < nnz; t += DL_THREADS) {
            const unsigned slot = sh.nz[t];
            tables[0].H01[slot] = make_double2(0.0, 0.0); tables[0].H23[slot] = make_double2(0.0, 0.0);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
        kept_total += __shfl_xor_sync(0xffffffffu, kept_total, o);
        binned_total += __shfl_xor_sync(0xffffffffu, binned_total, o);
        n_red += __shfl_xor_sync(0xffffffffu, n_red, o);
        conflicts += __shfl_xor_sync(0xffffffffu, conflicts, o);
    }
    if (lane == 0) {
        atomicAdd(&P.counters[2], evaluated);
        atomicAdd(&P.counters[5], kept_total);
        atomicAdd(&P.counters[6], binned_total);
        atomicAdd(&P.counters[7], n_red);
        if (CHECK && conflicts) atomicAdd(&P.counters[10], (unsigned long long)conflicts);
    }
}

}  // namespace
