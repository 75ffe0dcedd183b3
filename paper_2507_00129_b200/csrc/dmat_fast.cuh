// dmat_fast.cuh -- k_dmat_fast, the distortion-matrix kernel of the bucket-sorted forest-pair list
// (eqs. 2.6-2.7; the algebra T1..T4 is in dmat.cu's header).  Included by dmat.cu only.
//
// One warp per forest pair, forests staged from the padded catalogue.  Per forest pair:
//  windows  per row i of p the EXACT in-grid window [jlo, jhi) of q and the sign change jx
//           (lya_row_window) -- after this nothing has to re-test "inside the grid";
//  mask     stage 4 over the windows only: lanes over j, pure integer (pixel keys are staged), kept pairs
//           (about 1 % at f = 0.99) are queued as (i, j); sum (jhi - jlo) is the scanned-pair count;
//  pass A   the four H tables by the diagonal walk: lanes own diagonals d = j - i and HOLD the table
//           entry of their current run in registers (predicated release / acquire around one warp
//           barrier; no atomics).  One walk per side of chi_i = chi_j: the lanes of a row step then sit
//           on distinct r_par bins (q's spacing exceeds the bin width, lya_pair_key), so an entry has
//           one holder;
//  pass B   the non-zero table entries are compacted into a list;
//  pass C   drain: T1..T3 per kept pair over the row / column windows, T4 with lanes over the table
//           entries and an inner loop over the kept pairs; every update is one red.global.add.f64 into
//           the L2-resident Dn (transposed bin order).  T4 also clears the entries it read.
#pragma once
#include "lya_walk.cuh"

namespace {

constexpr int FD_WARPS = 15;                 // one CTA per SM (shared memory: 15.0 KB per warp)
constexpr int FD_THREADS = FD_WARPS * 32;
constexpr int FD_T = LYA_FAST_TILE;
constexpr int FD_ROWS = 16;
constexpr int FD_TP = ((FD_T + FD_ROWS - 1) / FD_ROWS) * FD_ROWS + 2;
constexpr int FD_PAD = 2;
constexpr int FD_TQ = FD_T + 2 * FD_PAD;
constexpr int FD_SLOTS = 306;                // (n_par + 1) * LYA_NCOL <= FD_SLOTS
constexpr int FD_KCAP = 48;                  // kept pairs queued per forest pair
constexpr int FD_KBATCH = 24;                // kept pairs drained together (coefficient tables)
constexpr int FD_CHUNK = 8;

struct DmFastParams {
    LyaPrep prep;
    const int32_t *pq;
    int64_t n_pairs;
    BinParams bp;
    unsigned long long seed, thr;
    double *Dn, *Wd;
    unsigned long long *counters;   // [4] next chunk, [2] evaluated, [3] error, [5] kept, [6] binned, [7] scatter-adds, [10] holder conflicts (CHECK)
};

struct DmKeysA { unsigned long long pk[FD_T], qk[FD_T]; };                 // mask scan: stage-4 keys of the pixels
struct DmDrainBC {                                                            // passes B and C
    double2 kc01[FD_KBATCH], kc23[FD_KBATCH];    // per kept pair of a batch: om (1, u_j), om (u_i, u_i u_j)
    unsigned short nz[FD_SLOTS];                 // non-zero slots
};
struct __align__(16) DmFastWarp {
    double2 H01[FD_SLOTS], H23[FD_SLOTS];    // (H_aa, H_ag), (H_ga, H_gg) per slot = col_rel * (n_par + 1) + row
    double2 pce[FD_TP];                      // (chi, ea) of p; rows >= len are sentinels
    double2 qce[FD_TQ];                      // (chi, ea) of q, FD_PAD sentinels either side
    double peg[FD_TP], qeg[FD_TQ];           // eg
    union { DmKeysA a; DmDrainBC b; } u;     // the keys are dead once the mask scan is done (shared memory buys occupancy)
    unsigned kept[FD_KCAP];                  // (A << 16) | (i << 8) | j   (A is filled in by the drain)
    unsigned char jlo[FD_T], jx[FD_T], jhi[FD_T];
};

// shared-memory ADDRESS of the H01 entry of a pixel pair in THIS walk (inside the grid and on the walk's
// side of chi_i = chi_j: sgn = 0 for chi_i >= chi_j, -1 otherwise); everything else -> the garbage entry.
// lim = min(LYA_NCOL, n_perp - c0).
template <bool POW2>
__device__ __forceinline__ unsigned dm_key(const BinParams &bp, const PairBin &g, double chi_i, double chi_j, unsigned c0,
                                           unsigned lim, unsigned np1, int sgn, unsigned h01, unsigned garbage)
{
    const double d = __dsub_rn(chi_i, chi_j);
    const double t = __dadd_rn(chi_i, chi_j);
    unsigned bx, by;
    if (POW2) {
        bx = lya_floor_u32(__dmul_rn(fabs(d), g.cx));
        by = lya_floor_u32(__dmul_rn(t, g.sy));
    } else {
        const double rpar = __dmul_rn(fabs(d), g.c), rperp = __dmul_rn(t, g.s);
        bx = (rpar < bp.rpar_max) ? min(lya_floor_u32(__dmul_rn(rpar, bp.inv_par)), (unsigned)(bp.n_par - 1)) : (unsigned)bp.n_par;
        by = (rperp < bp.rperp_max) ? min(lya_floor_u32(__dmul_rn(rperp, bp.inv_perp)), (unsigned)(bp.n_perp - 1)) : 0x7fffffffu;
    }
    const unsigned col = by - c0;
    const bool valid = ((__double2hiint(d) ^ sgn) >= 0) & (bx < np1 - 1u) & (col < lim);
    return valid ? h01 + ((col * np1 + bx) << 4) : garbage;
}

// pass A over rows [r0, r1] (a multiple of D rows; rows >= len are sentinels) and diagonals [dlo, dhi].
// `key`/`cur` are shared-memory addresses of H01 entries; H23 sits at a fixed offset.
template <int D, bool POW2, bool CHECK>
__device__ __forceinline__ void dm_walk(DmFastWarp &ws, unsigned h01, int r0, int r1, int mq, int dlo, int dhi,
                                        int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned lim, unsigned np1,
                                        int lane, unsigned long long &evaluated, unsigned &conflicts)
{
    constexpr unsigned H23OFF = (unsigned)(sizeof(double2) * FD_SLOTS);
    const double2 *qce = ws.qce + FD_PAD;
    const double *qeg = ws.qeg + FD_PAD;
    const unsigned garbage = h01 + ((np1 - 1u) << 4);
    for (int d0 = dlo; d0 <= dhi; d0 += 32 * D) {
        const int dl = d0 + lane * D;
        unsigned cur[D], key[D];
        double h0[D], h1[D], h2[D], h3[D], fa[D], fg[D];
        double wc[D], wa[D], wg[D];                         // sliding window over q: chi, ea, eg
        double pa_c, pg_c;
#pragma unroll
        for (int k = 0; k < D; ++k) { cur[k] = garbage; h0[k] = 0.0; h1[k] = 0.0; h2[k] = 0.0; h3[k] = 0.0; }
#pragma unroll
        for (int k = 0; k < D; ++k) {
            const int j = min(max(r0 + dl + k, -FD_PAD), mq + FD_PAD - 1);
            const double2 v = qce[j];
            wc[k] = v.x; wa[k] = v.y; wg[k] = qeg[j];
        }
        {
            const double2 pv = ws.pce[r0];
#pragma unroll
            for (int k = 0; k < D; ++k) {
                key[k] = dm_key<POW2>(bp, g, pv.x, wc[k], c0, lim, np1, sgn, h01, garbage);
                fa[k] = wa[k]; fg[k] = wg[k];
            }
            pa_c = pv.y; pg_c = ws.peg[r0];
        }
        evaluated += (unsigned long long)(r1 - r0 + 1) * D;
        for (int ib = r0; ib <= r1; ib += D) {
#pragma unroll
            for (int u = 0; u < D; ++u) {
                const int i = ib + u;                       // window slot of q[i + dl + k] is (k + u) % D
                bool ch[D];
                if (CHECK) {                                // invariant: a non-garbage entry has one holder (debug runs only)
                    for (int src = 0; src < 32; ++src)
#pragma unroll
                        for (int k2 = 0; k2 < D; ++k2) {
                            const unsigned other = __shfl_sync(0xffffffffu, key[k2], src);
#pragma unroll
                            for (int k = 0; k < D; ++k)
                                if (other == key[k] && key[k] != garbage && (src < lane || (src == lane && k2 < k))) conflicts += 1u;
                        }
                }
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    ch[k] = key[k] != cur[k];
                    sts_v2_if(ch[k], cur[k], h0[k], h1[k]);                             // release
                    sts_v2_if(ch[k], cur[k] + H23OFF, h2[k], h3[k]);
                }
                __syncwarp();
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    lds_v2_if(ch[k], key[k], h0[k], h1[k]);                             // acquire
                    lds_v2_if(ch[k], key[k] + H23OFF, h2[k], h3[k]);
                    cur[k] = key[k];
                }
                // row i + 1: its new q pixel replaces q[i + dl] in window slot u
                unsigned key_n[D];
                double fa_n[D], fg_n[D];
                {
                    const int j = min(max(i + dl + D, -FD_PAD), mq + FD_PAD - 1);
                    const double2 v = qce[j];
                    wc[u] = v.x; wa[u] = v.y; wg[u] = qeg[j];
                }
                const double2 pv = ws.pce[i + 1];
                const double pg_n = ws.peg[i + 1];
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    const int sl = (k + u + 1) % D;
                    key_n[k] = dm_key<POW2>(bp, g, pv.x, wc[sl], c0, lim, np1, sgn, h01, garbage);
                    fa_n[k] = wa[sl]; fg_n[k] = wg[sl];
                }
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    h0[k] = fma(pa_c, fa[k], h0[k]); h1[k] = fma(pa_c, fg[k], h1[k]);
                    h2[k] = fma(pg_c, fa[k], h2[k]); h3[k] = fma(pg_c, fg[k], h3[k]);
                    fa[k] = fa_n[k]; fg[k] = fg_n[k]; key[k] = key_n[k];
                }
                pa_c = pv.y; pg_c = pg_n;
            }
        }
#pragma unroll
        for (int k = 0; k < D; ++k) {
            sts_v2_if(true, cur[k], h0[k], h1[k]);
            sts_v2_if(true, cur[k] + H23OFF, h2[k], h3[k]);
        }
        __syncwarp();
    }
}

template <bool POW2, bool CHECK>
__device__ __forceinline__ void dm_walk_any(DmFastWarp &ws, unsigned h01, int r0, int r1, int mq, int dlo, int dhi,
                                            int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned lim, unsigned np1,
                                            int lane, unsigned long long &evaluated, unsigned &conflicts)
{
    if (dhi < dlo) return;
    const int nd = dhi - dlo + 1;
    if (nd <= 32) dm_walk<1, POW2, CHECK>(ws, h01, r0, r1, mq, dlo, dhi, sgn, bp, g, c0, lim, np1, lane, evaluated, conflicts);
    else dm_walk<2, POW2, CHECK>(ws, h01, r0, r1, mq, dlo, dhi, sgn, bp, g, c0, lim, np1, lane, evaluated, conflicts);
}

// pass C: drain n queued kept pairs (kept[e] = (i << 8) | j on entry; the bin A is OR-ed into bits 16.. here).
// clear: T4 zeroes the table entries it read (last batch of a forest pair).
template <bool POW2>
__device__ __forceinline__ void dm_drain_batch(DmFastWarp &ws, unsigned *kept, int n, int nnz, int mp, const DmFastParams &P,
                                               const PairBin &g, int c0, long long offp, long long offq, int lane,
                                               bool clear, unsigned long long &n_red)
{
    const BinParams &bp = P.bp;
    const int nb = bp.n_par * bp.n_perp, np1 = bp.n_par + 1;
    const double2 *qce = ws.qce + FD_PAD;
    const double *qeg = ws.qeg + FD_PAD;
    // coefficients of every kept pair (lanes over kept pairs) and T1: Dn[A][A] += om, Wd[A] += om
    for (int e = lane; e < n; e += 32) {
        const unsigned rec = kept[e];
        const int i = (rec >> 8) & 0xff, j = rec & 0xff;
        const int A = lya_pix_bin_t<POW2>(bp, g, ws.pce[i].x, qce[j].x);           // inside the grid by construction
        const double om = P.prep.w[offp + i] * P.prep.w[offq + j], ui = P.prep.u[offp + i], uj = P.prep.u[offq + j];
        const double omi = om * ui;
        ws.u.b.kc01[e] = make_double2(om, om * uj);
        ws.u.b.kc23[e] = make_double2(omi, omi * uj);
        kept[e] = ((unsigned)A << 16) | (rec & 0xffffu);
        atomicAdd(P.Dn + (size_t)A * nb + A, om);
        atomicAdd(P.Wd + A, om);
        n_red += 2;
    }
    __syncwarp();
    // T2: -(om ea_j' + om u_j eg_j') over row i's window;  T3: -(om ea_i' + om u_i eg_i') over the rows whose
    // window holds j.  The windows are exact, so no pair is re-tested against the grid.
    for (int e = 0; e < n; ++e) {
        const unsigned rec = kept[e];
        const int i = (rec >> 8) & 0xff, j = rec & 0xff;
        const double2 c01 = ws.u.b.kc01[e], c23 = ws.u.b.kc23[e];
        const double ci = ws.pce[i].x, cj = qce[j].x;
        double *row = P.Dn + (size_t)(rec >> 16) * nb;
        const int jl = ws.jlo[i], jh = ws.jhi[i];
        for (int j2 = jl + lane; j2 < jh; j2 += 32) {
            const double2 q2 = qce[j2];
            const int B = lya_pix_bin_t<POW2>(bp, g, ci, q2.x);
            atomicAdd(row + B, -fma(c01.y, qeg[j2], c01.x * q2.y));
        }
        n_red += (unsigned long long)(lane == 0 ? jh - jl : 0);
        for (int i2 = lane; i2 < mp; i2 += 32) {
            if (j >= (int)ws.jlo[i2] && j < (int)ws.jhi[i2]) {
                const double2 p2 = ws.pce[i2];
                const int B = lya_pix_bin_t<POW2>(bp, g, p2.x, cj);
                atomicAdd(row + B, -fma(c23.x, ws.peg[i2], c01.x * p2.y));
                n_red += 1;
            }
        }
    }
    // T4: lanes over the non-zero table entries, inner loop over the kept pairs
    for (int t = lane; t < nnz; t += 32) {
        const int slot = ws.u.b.nz[t];
        const int cr = slot / np1, bx = slot - cr * np1;
        double *colB = P.Dn + ((c0 + cr) * bp.n_par + bx);
        const double2 a = ws.H01[slot], b = ws.H23[slot];
        if (clear) { ws.H01[slot] = make_double2(0.0, 0.0); ws.H23[slot] = make_double2(0.0, 0.0); }
#pragma unroll 2
        for (int e = 0; e < n; ++e) {
            const unsigned A = kept[e] >> 16;
            const double2 c01 = ws.u.b.kc01[e], c23 = ws.u.b.kc23[e];
            const double v = fma(c23.y, b.y, fma(c23.x, b.x, fma(c01.y, a.y, c01.x * a.x)));
            atomicAdd(colB + (size_t)A * nb, v);
        }
        n_red += (unsigned long long)n;
    }
}

template <bool POW2, bool CHECK>
__global__ void __launch_bounds__(FD_THREADS, 1) k_dmat_fast(DmFastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    DmFastWarp &ws = ((DmFastWarp *)smem_raw)[wid];
    const BinParams bp = P.bp;
    const unsigned np1 = (unsigned)bp.n_par + 1u;
    const int n_slots = (int)np1 * LYA_NCOL;
    for (int t = lane; t < FD_SLOTS; t += 32) { ws.H01[t] = make_double2(0.0, 0.0); ws.H23[t] = make_double2(0.0, 0.0); }
    if (lane < FD_PAD) { ws.qce[lane] = make_double2(LYA_CHI_SENTINEL, 0.0); ws.qeg[lane] = 0.0; }
    __syncwarp();
    const double2 *qce = ws.qce + FD_PAD;
    const unsigned h01 = (unsigned)__cvta_generic_to_shared(ws.H01);
    unsigned long long evaluated = 0, kept_total = 0, binned_total = 0, n_red = 0;
    unsigned conflicts = 0;
    int cur_p = -1, head_p = -1;
    ForestHead hp;
    hp.len = 0;
    const int64_t n_chunks = (P.n_pairs + FD_CHUNK - 1) / FD_CHUNK;
    for (;;) {
        unsigned long long chunk = 0;
        if (lane == 0) chunk = atomicAdd(&P.counters[4], 1ull);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if ((int64_t)chunk >= n_chunks) break;
        const int64_t k0 = (int64_t)chunk * FD_CHUNK, k1 = min(k0 + FD_CHUNK, P.n_pairs);
        for (int64_t k = k0; k < k1; ++k) {
            const int2 e = ((const int2 *)P.pq)[k];
            const int p = e.x, q = e.y;
            if (p != head_p) { hp = P.prep.head[p]; head_p = p; }
            const ForestHead hq = P.prep.head[q];
            const int mp = hp.len, mq = hq.len;
            if ((hp.flags | hq.flags) & 1) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_DEGENERATE);
                continue;
            }
            double s, c;
            lya_pair_sc(hp.ux, hp.uy, hp.uz, hq.ux, hq.uy, hq.uz, s, c);
            const PairBin g = lya_make_pairbin(bp, s, c);
            int c0;
            const int key = lya_pair_key<POW2>(bp, g, hp, hq, c0);
            if (key >= bp.n_perp) continue;                  // cannot happen in the fast range
            const unsigned lim = (unsigned)min(LYA_NCOL, bp.n_perp - c0);
            __syncwarp();
            // ---- stage p (when it changes) and q: (chi, ea) pairs with 16-byte loads, eg, stage-4 keys ----
            if (p != cur_p) {
                const double2 *sce = P.prep.ce + hp.off;
                const double2 *sg = (const double2 *)(P.prep.eg + hp.off);
                for (int t = lane; t < mp; t += 32) ws.pce[t] = sce[t];
                for (int t = lane; 2 * t < mp; t += 32) ((double2 *)ws.peg)[t] = sg[t];
                __syncwarp();
                for (int t = mp + lane; t < FD_TP; t += 32) {            // sentinel rows (!= q's sentinel: r_par never 0)
                    ws.pce[t] = make_double2(2.0 * LYA_CHI_SENTINEL, 0.0); ws.peg[t] = 0.0;
                }
                cur_p = p;
            }
            {
                const double2 *sce = P.prep.ce + hq.off;
                const double2 *sg = (const double2 *)(P.prep.eg + hq.off);
                const int npad = (mq + 1) & ~1;
                for (int t = lane; t < npad; t += 32) ws.qce[FD_PAD + t] = sce[t];       // (the pad pixel of an odd forest is a sentinel)
                for (int t = lane; 2 * t < npad; t += 32) ((double2 *)(ws.qeg + FD_PAD))[t] = sg[t];
                for (int t = lane; t < mq; t += 32) ws.u.a.qk[t] = lya_key_hi(P.seed, (unsigned long long)(hq.pix0 + t));
                // (the keys share their storage with the drain tables, so p's keys are rebuilt for every pair)
                for (int t = lane; t < mp; t += 32) ws.u.a.pk[t] = lya_key_lo(P.seed, (unsigned long long)(hp.pix0 + t));
                if (lane < FD_PAD) {
                    const int j = FD_PAD + npad + lane;
                    ws.qce[j] = make_double2(LYA_CHI_SENTINEL, 0.0); ws.qeg[j] = 0.0;
                }
            }
            __syncwarp();
            // ---- windows: per row of p the exact in-grid window [jlo, jhi) of q and the sign change jx ----
            const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;
            const double Tchi = (s > 0.0) ? (bp.rperp_max / s) * (1.0 + 1e-12) + 1e-9 : 1e300;
            for (int i = lane; i < mp; i += 32) {
                int jlo, jx, jhi;
                lya_row_window<POW2>(bp, g, qce, mq, ws.pce[i].x, R, Tchi, jlo, jx, jhi);
                ws.jlo[i] = (unsigned char)jlo; ws.jx[i] = (unsigned char)jx; ws.jhi[i] = (unsigned char)jhi;
            }
            __syncwarp();
            // ---- mask: stage 4 over the windows (integer only); queue the kept pairs ----
            unsigned nk = 0, binned = 0;
            for (int i = 0; i < mp; ++i) {
                const int jl = ws.jlo[i], jh = ws.jhi[i];
                const unsigned long long pki = ws.u.a.pk[i];
                binned += (unsigned)(jh - jl);
                for (int j0 = jl; j0 < jh; j0 += 32) {
                    const int j = j0 + lane;
                    const bool kp = (j < jh) && lya_keep_pair(pki, ws.u.a.qk[min(j, FD_T - 1)], P.thr);
                    const unsigned bal = __ballot_sync(0xffffffffu, kp);
                    if (bal) {
                        const unsigned idx = nk + __popc(bal & ((1u << lane) - 1u));
                        if (kp && idx < FD_KCAP) ws.kept[idx] = ((unsigned)i << 8) | (unsigned)j;
                        nk += __popc(bal);
                    }
                }
            }
            binned_total += binned; kept_total += nk;
            // ---- pass A: H tables ----
            for (int i0 = 0; i0 < mp; i0 += FD_ROWS) {
                const int i = i0 + lane;
                int plo = 1 << 20, phi = -(1 << 20), nlo = 1 << 20, nhi = -(1 << 20);
                int pr0 = 1 << 20, pr1 = -1, nr0 = 1 << 20, nr1 = -1;
                if (lane < FD_ROWS && i < mp) {
                    const int jl = ws.jlo[i], jh = ws.jhi[i], jx = ws.jx[i];
                    if (jx > jl) { plo = jl - i; phi = jx - 1 - i; pr0 = i; pr1 = i; }
                    if (jh > jx) { nlo = jx - i; nhi = jh - 1 - i; nr0 = i; nr1 = i; }
                }
                plo = __reduce_min_sync(0xffffffffu, plo); phi = __reduce_max_sync(0xffffffffu, phi);
                nlo = __reduce_min_sync(0xffffffffu, nlo); nhi = __reduce_max_sync(0xffffffffu, nhi);
                pr0 = __reduce_min_sync(0xffffffffu, pr0); pr1 = __reduce_max_sync(0xffffffffu, pr1);
                nr0 = __reduce_min_sync(0xffffffffu, nr0); nr1 = __reduce_max_sync(0xffffffffu, nr1);
#pragma unroll 1
                for (int sgn = 0; sgn >= -1; --sgn) {       // one call site: chi_i >= chi_j, then chi_i < chi_j
                    const int r0 = sgn ? nr0 : pr0, r1 = sgn ? nr1 : pr1;
                    if (r1 < r0) continue;
                    dm_walk_any<POW2, CHECK>(ws, h01, r0 & ~1, r1 | 1, mq, sgn ? nlo : plo, sgn ? nhi : phi, sgn, bp, g,
                                             (unsigned)c0, lim, np1, lane, evaluated, conflicts);
                }
            }
            __syncwarp();
            // ---- pass B: compact the non-zero entries (H_aa > 0 wherever a pair with weight fell) ----
            int nnz = 0;
            for (int t0 = 0; t0 < n_slots; t0 += 32) {
                const int t = t0 + lane;
                bool nzf = false;
                if (t < n_slots) {
                    const int cr = t / (int)np1, bx = t - cr * (int)np1;
                    const double2 a = ws.H01[t], b = ws.H23[t];
                    nzf = (bx < bp.n_par) && (a.x != 0.0 || a.y != 0.0 || b.x != 0.0 || b.y != 0.0);
                }
                const unsigned bal = __ballot_sync(0xffffffffu, nzf);
                if (nzf) ws.u.b.nz[nnz + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)t;
                nnz += __popc(bal);
            }
            __syncwarp();
            // ---- pass C (one drain call site: the kernel's code has to stay small for the instruction cache) ----
            // Normally the queue holds every kept pair.  With more kept pairs than the queue holds (small
            // reject fractions) the mask is redone row by row and the queue drained each time it fills.
            const bool overflow = nk > FD_KCAP;
            int n_q = overflow ? 0 : (int)nk;
            int si = 0, sj = (overflow && mp > 0) ? (int)ws.jlo[0] : 0;
            for (;;) {
                bool done = true;
                if (overflow) {
                    while (si < mp) {
                        const int jh = ws.jhi[si];
                        if (sj >= jh) { ++si; sj = (si < mp) ? (int)ws.jlo[si] : 0; continue; }
                        const int j = sj + lane;
                        const bool kp = (j < jh) && lya_keep_pair(lya_key_lo(P.seed, (unsigned long long)(hp.pix0 + si)),
                                                                  lya_key_hi(P.seed, (unsigned long long)(hq.pix0 + j)), P.thr);   // (the staged keys are gone)
                        const unsigned bal = __ballot_sync(0xffffffffu, kp);
                        if (n_q + __popc(bal) > FD_KCAP) break;          // drain first, then redo these 32 pixels
                        if (kp) ws.kept[n_q + __popc(bal & ((1u << lane) - 1u))] = ((unsigned)si << 8) | (unsigned)j;
                        n_q += __popc(bal);
                        sj += 32;
                    }
                    done = si >= mp;
                }
                __syncwarp();
                for (int e0 = 0; e0 < n_q || e0 == 0; e0 += FD_KBATCH) {
                    const int nb_e = min(FD_KBATCH, n_q - e0);
                    dm_drain_batch<POW2>(ws, ws.kept + e0, nb_e, nnz, mp, P, g, c0, hp.off, hq.off, lane,
                                         done && e0 + FD_KBATCH >= n_q, n_red);
                    __syncwarp();
                }
                if (done) break;
                n_q = 0;
            }
            // the garbage entry collects every out-of-grid product: clear it too
            if (lane == 0) { ws.H01[np1 - 1u] = make_double2(0.0, 0.0); ws.H23[np1 - 1u] = make_double2(0.0, 0.0); }
            __syncwarp();
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
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
