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

// Two size classes of the same kernel (template parameter CLS):
//   class 0: forests of up to LYA_FAST_TILE (72) pixels -- the BASELINE configs; 15 warps per SM;
//   class 1: forests of up to LYA_FAST_TILE2 (144) pixels -- native-resolution shapes (DESIGN.md NEXT-3): longer
//            staging tiles and kept-pair queue, 11 warps per SM (what its 20.5 KB per warp allow).
// In both, pass A takes a DIAGONAL STRIDE ds: a pass covers the diagonals d0 + ds * lane, so the lanes of a row
// step sit ds pixels of q apart; ds is the smallest integer with ds * (q's pixel spacing) > r_par bin width, which
// keeps "one holder per table entry" true when the pixels are finer than the bins (ds passes, one per residue,
// cover every diagonal; the number of lane-slots walked is the same).
#ifndef LYA_FD_WARPS
#define LYA_FD_WARPS 15
#endif
#ifndef LYA_FD_WARPS2
#define LYA_FD_WARPS2 11
#endif
template <int CLS> struct DmCfg;
template <> struct DmCfg<0> { static constexpr int T = LYA_FAST_TILE, WARPS = LYA_FD_WARPS, KCAP = 48; };
template <> struct DmCfg<1> { static constexpr int T = LYA_FAST_TILE2, WARPS = LYA_FD_WARPS2, KCAP = 192; };
// (the FD_* names below depend on the template parameter CLS of the struct / function they are used in)
#define FD_WARPS (DmCfg<CLS>::WARPS)         // one CTA per SM; private shared memory per warp + the table pool
#define FD_THREADS (DmCfg<CLS>::WARPS * 32)
#define FD_T (DmCfg<CLS>::T)
#define FD_TP (((DmCfg<CLS>::T + 15) / 16) * 16 + 2)
#define FD_TQ (DmCfg<CLS>::T + 2 * FD_PAD)
#define FD_KCAP (DmCfg<CLS>::KCAP)           // kept pairs queued per forest pair
#define FD_RPL ((DmCfg<CLS>::T + 31) / 32)   // rows of p per lane in the mask scan's prefix sum
constexpr int FD_SMEM_MAX = 232448;          // 227 KB: the most a CTA can have on sm_100
#ifndef LYA_FD_ROWS
#define LYA_FD_ROWS 16
#endif
constexpr int FD_ROWS = LYA_FD_ROWS;         // rows of p per pass-A group
constexpr int FD_PAD = 2;
constexpr int FD_SLOTS = 302;                // n_par * LYA_NCOL + 1 <= FD_SLOTS (the last slot used is garbage)
constexpr int FD_KBATCH = 24;                // kept pairs drained together (coefficient tables)
#ifndef LYA_FD_CHUNK
#define LYA_FD_CHUNK 8
#endif
constexpr int FD_CHUNK = LYA_FD_CHUNK;    // forest pairs claimed per atomic
constexpr int FD_DS_MAX = 8;                 // largest diagonal stride the fast kernel takes
// Profiling aids (compile-time, off by default; results are WRONG with any of them): -DLYA_ABL_NO_T23,
// -DLYA_ABL_NO_T4, -DLYA_ABL_NO_MASK, -DLYA_ABL_NO_WALK drop one phase so that its share of the kernel time can
// be measured as a difference (profiles/r2*_dmat_ablation.md).

struct DmFastParams {
    LyaPrep prep;
    const int32_t *pq;
    int64_t n_pairs;
    BinParams bp;
    unsigned long long seed, thr;
    double *Dn, *Wd;
    unsigned long long *counters;   // [4] next chunk, [2] evaluated, [3] error, [5] kept, [6] binned, [7] scatter-adds, [10] holder conflicts (CHECK)
};

template <int CLS> struct DmKeysA {                                          // mask scan
    unsigned long long qk[FD_T], pk[FD_T];       // stage-4 keys of the pixels of q and p
    unsigned short pre[FD_T + 2];                // pre[i] = in-window pairs of the rows before i
};
struct DmDrainBC {                                                            // passes B and C
    double2 kc01[FD_KBATCH], kc23[FD_KBATCH];    // per kept pair of a batch: om (1, u_j), om (u_i, u_i u_j)
    unsigned short nz[FD_SLOTS];                 // non-zero slots
};
// H tables live in a POOL shared by the warps of the CTA (a warp holds one from pass A to the end of T4; a free
// table is all zero).  With as many tables as warps (the default) nobody ever waits; fewer tables than warps
// were measured to lose more to waiting than extra warps bring (profiles/r2b_dmat_ablation.md).
struct __align__(16) DmTable {
    double2 H01[FD_SLOTS], H23[FD_SLOTS];    // (H_aa, H_ag), (H_ga, H_gg) per slot = col_rel * n_par + b_par; slot LYA_NCOL * n_par = garbage
};
template <int CLS> struct __align__(16) DmFastWarp {
    double2 pce[FD_TP];                      // (chi, ea) of p; rows >= len are sentinels
    double2 qce[FD_TQ];                      // (chi, ea) of q, FD_PAD sentinels either side
    double peg[FD_TP], qeg[FD_TQ];           // eg
    union { DmKeysA<CLS> a; DmDrainBC b; } u;     // the keys are dead once the mask scan is done (shared memory buys occupancy)
    unsigned kept[FD_KCAP];                  // (A << 16) | (i << 8) | j   (A is filled in by the drain)
    unsigned char jlo[FD_T + 4], jx[FD_T + 4], jhi[FD_T + 4];   // (row len = a stop row for the mask scan)
    unsigned nkept, pad_[1];
};
constexpr int FD_POOL_HDR = 128;             // owner flags of the tables (one int each)
template <int CLS> struct DmPool {
    static constexpr int FIT = (FD_SMEM_MAX - FD_POOL_HDR - (int)sizeof(DmFastWarp<CLS>) * FD_WARPS) / (int)sizeof(DmTable);
#ifdef LYA_FD_NTABLES
    static constexpr int NTABLES = LYA_FD_NTABLES;
#else
    static constexpr int NTABLES = FIT < FD_WARPS ? FIT : FD_WARPS;
#endif
    static constexpr size_t SMEM_BYTES = FD_POOL_HDR + sizeof(DmTable) * NTABLES + sizeof(DmFastWarp<CLS>) * FD_WARPS;
    static_assert(NTABLES >= 2 && NTABLES * 4 <= FD_POOL_HDR && SMEM_BYTES <= (size_t)FD_SMEM_MAX, "table pool");
};
#define FD_NTABLES (DmPool<CLS>::NTABLES)

// shared-memory ADDRESS of the H01 entry of a pixel pair in THIS walk (inside the grid and on the walk's
// side of chi_i = chi_j: sgn = 0 for chi_i >= chi_j, -1 otherwise); everything else -> the garbage entry.
// lim = min(LYA_NCOL, n_perp - c0).  The slot col * n_par + b_par is also the pair's offset from the first
// bin of column c0 in the transposed bin order of Dn.
template <bool POW2>
__device__ __forceinline__ unsigned dm_key(const BinParams &bp, const PairBin &g, double chi_i, double chi_j, unsigned c0,
                                           unsigned lim, unsigned npar, int sgn, unsigned h01, unsigned garbage)
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
    const unsigned addr = h01 + ((col * npar + bx) << 4);
    unsigned key;
    asm("{\n .reg .pred v;\n setp.ge.s32 v, %1, 0;\n setp.lt.and.u32 v, %2, %3, v;\n setp.lt.and.u32 v, %4, %5, v;\n"
        " selp.u32 %0, %6, %7, v;\n}"
        : "=r"(key) : "r"(__double2hiint(d) ^ sgn), "r"(bx), "r"(npar), "r"(col), "r"(lim), "r"(addr), "r"(garbage));
    return key;
}

// pass A over rows [r0, r1] (a multiple of D rows; rows >= len are sentinels) and diagonals [dlo, dhi].
// `key`/`cur` are shared-memory addresses of H01 entries; H23 sits at a fixed offset.
// (WS: the staging area -- pce, peg, qce, qeg -- of a warp, DmFastWarp, or of a CTA, dmat_long.cuh)
template <int D, bool POW2, bool CHECK, class WS>
__device__ __forceinline__ void dm_walk(WS &ws, unsigned h01, int r0, int r1, int mq, int dlo, int dhi, int ds,
                                        int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned lim, unsigned npar,
                                        int lane, unsigned long long &evaluated, unsigned &conflicts)
{
    constexpr unsigned H23OFF = (unsigned)(sizeof(double2) * FD_SLOTS);     // DmTable: H23 follows H01
    const double2 *qce = ws.qce + FD_PAD;
    const double *qeg = ws.qeg + FD_PAD;
    const unsigned garbage = h01 + ((npar * LYA_NCOL) << 4);
    // D == 1: blocks of 32 * ds diagonals, ds passes per block (one per residue), lane l on diagonal d0 + ds * l;
    // D == 2 (ds == 1 only): blocks of 64 diagonals, lane l on diagonals d0 + 2 l and d0 + 2 l + 1.
    const int step = (D == 1) ? ds : D, n_res = (D == 1) ? ds : 1;
    const int n_pass = ((dhi - dlo) / (32 * step) + 1) * n_res;
    for (int pass = 0; pass < n_pass; ++pass) {
        const int d0 = dlo + (pass / n_res) * (32 * step) + pass % n_res;
        if (d0 > dhi) continue;
        const int dl = d0 + lane * step;
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
                key[k] = dm_key<POW2>(bp, g, pv.x, wc[k], c0, lim, npar, sgn, h01, garbage);
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
                    // (one unsigned min clamps both ends: a negative index wraps to the right-hand sentinel)
                    const unsigned j = min((unsigned)(i + dl + D + FD_PAD), (unsigned)(mq + 2 * FD_PAD - 1));
                    const double2 v = ws.qce[j];
                    wc[u] = v.x; wa[u] = v.y; wg[u] = ws.qeg[j];
                }
                const double2 pv = ws.pce[i + 1];
                const double pg_n = ws.peg[i + 1];
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    const int sl = (k + u + 1) % D;
                    key_n[k] = dm_key<POW2>(bp, g, pv.x, wc[sl], c0, lim, npar, sgn, h01, garbage);
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

template <bool POW2, bool CHECK, class WS>
__device__ __forceinline__ void dm_walk_any(WS &ws, unsigned h01, int r0, int r1, int mq, int dlo, int dhi, int ds,
                                            int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned lim, unsigned npar,
                                            int lane, unsigned long long &evaluated, unsigned &conflicts)
{
    if (dhi < dlo) return;
    const int nd = dhi - dlo + 1;
    if (nd <= 32 || ds > 1) dm_walk<1, POW2, CHECK>(ws, h01, r0, r1, mq, dlo, dhi, ds, sgn, bp, g, c0, lim, npar, lane, evaluated, conflicts);
    else dm_walk<2, POW2, CHECK>(ws, h01, r0, r1, mq, dlo, dhi, 1, sgn, bp, g, c0, lim, npar, lane, evaluated, conflicts);
}

// transposed bin index b_perp * n_par + b_par of a pixel pair KNOWN to be inside the grid (exact windows)
template <bool POW2>
__device__ __forceinline__ int dm_bin_in(const BinParams &bp, const PairBin &g, double chi_i, double chi_j)
{
    const double d = __dsub_rn(chi_i, chi_j);
    const double t = __dadd_rn(chi_i, chi_j);
    unsigned bx, by;
    if (POW2) {
        bx = lya_floor_u32(__dmul_rn(fabs(d), g.cx));
        by = lya_floor_u32(__dmul_rn(t, g.sy));
    } else {
        bx = min(lya_floor_u32(__dmul_rn(__dmul_rn(fabs(d), g.c), bp.inv_par)), (unsigned)(bp.n_par - 1));
        by = min(lya_floor_u32(__dmul_rn(__dmul_rn(t, g.s), bp.inv_perp)), (unsigned)(bp.n_perp - 1));
    }
    return (int)(by * (unsigned)bp.n_par + bx);
}

__device__ __forceinline__ void dm_red(double *addr, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" :: "l"(addr), "d"(v) : "memory");
}


// ---- pass C, first half (no H table needed) ------------------------------------------------------
// n queued kept pairs, kept[e] = (i << 8) | j on entry.  Coefficients of every kept pair into kc01 / kc23, the
// bin A OR-ed into bits 16.. of kept[e]; with scatter: T1 (Dn[A][A] += om, Wd[A] += om), T2 (row i's window)
// and T3 (the rows whose window holds j).  The windows are exact, so no pair is re-tested against the grid.
// Dn has n_bins^2 <= 2^24 entries, so element indices are 32-bit and an address is one IMAD.WIDE away.
// (Tried and dropped: keeping each lane's rows / columns in registers for the whole drain -- fewer shared-memory
// wavefronts, but the extra live registers spilled and it was 3-9 % slower.)
template <bool POW2, int CLS>
__device__ __forceinline__ void dm_drain_t123(DmFastWarp<CLS> &ws, unsigned *kept, int n, int mp, const DmFastParams &P,
                                              const PairBin &g, long long offp, long long offq, int lane,
                                              bool scatter, unsigned &n_red)
{
    const BinParams &bp = P.bp;
    const unsigned nb = (unsigned)(bp.n_par * bp.n_perp);
    const double2 *qce = ws.qce + FD_PAD;
    const double *qeg = ws.qeg + FD_PAD;
    double *const Dn = P.Dn;
    for (int e = lane; e < n; e += 32) {
        const unsigned rec = kept[e];
        const int i = (rec >> 8) & 0xff, j = rec & 0xff;
        const unsigned A = (unsigned)dm_bin_in<POW2>(bp, g, ws.pce[i].x, qce[j].x);
        const double om = P.prep.w[offp + i] * P.prep.w[offq + j], ui = P.prep.u[offp + i], uj = P.prep.u[offq + j];
        const double omi = om * ui;
        ws.u.b.kc01[e] = make_double2(om, om * uj);
        ws.u.b.kc23[e] = make_double2(omi, omi * uj);
        kept[e] = (A << 16) | (rec & 0xffffu);
        if (scatter) {
            dm_red(Dn + (A * nb + A), om);
            dm_red(P.Wd + A, om);
            n_red += 2u;
        }
    }
    __syncwarp();
    if (!scatter) return;
#ifdef LYA_ABL_NO_T23
    return;
#endif
#pragma unroll 1
    for (int e = 0; e < n; ++e) {
        const unsigned rec = kept[e];
        const int i = (rec >> 8) & 0xff, j = rec & 0xff;
        const double2 c01 = ws.u.b.kc01[e];
        const double m0 = -c01.x, m1 = -c01.y, m2 = -ws.u.b.kc23[e].x;
        const double ci = ws.pce[i].x, cj = qce[j].x;
        const unsigned row = (rec >> 16) * nb;
        const int jh = ws.jhi[i];
        // T2 and T3 with the 32-wide blocks of the row window / of the rows unrolled: the window tests of every block
        // are issued before the first body, and there is no loop bookkeeping
        {
            const int j20 = ws.jlo[i] + lane;
            bool in3[FD_RPL];
#pragma unroll
            for (int k = 0; k < FD_RPL; ++k) {
                const int i2 = lane + 32 * k;
                in3[k] = false;
                if (i2 < mp) { const unsigned lo2 = ws.jlo[i2]; in3[k] = (unsigned)j - lo2 < (unsigned)ws.jhi[i2] - lo2; }
            }
#pragma unroll
            for (int k = 0; k < FD_RPL; ++k) {                                       // T2
                const int j2 = j20 + 32 * k;
                if (j2 < jh) {
                    const double2 q2 = qce[j2];
                    dm_red(Dn + (row + (unsigned)dm_bin_in<POW2>(bp, g, ci, q2.x)), fma(m1, qeg[j2], m0 * q2.y));
                    n_red += 1u;
                }
            }
#pragma unroll
            for (int k = 0; k < FD_RPL; ++k) {                                       // T3
                const int i2 = lane + 32 * k;
                if (in3[k]) {
                    const double2 p2 = ws.pce[i2];
                    dm_red(Dn + (row + (unsigned)dm_bin_in<POW2>(bp, g, p2.x, cj)), fma(m2, ws.peg[i2], m0 * p2.y));
                    n_red += 1u;
                }
            }
        }
    }
}

// ---- pass C, second half: T4 of n kept pairs whose coefficients are in kc01 / kc23: lanes over the non-zero
// table entries (consecutive slots are consecutive bins of Dn's row), kept pairs EIGHT at a time with their
// coefficients in registers.  wipe: zero the table entries read (last use of the table for this forest pair).
#ifndef LYA_FD_T4B
#define LYA_FD_T4B 4
#endif
constexpr int FD_T4B = LYA_FD_T4B;
template <int CLS>
__device__ __forceinline__ void dm_drain_t4(DmFastWarp<CLS> &ws, DmTable &tb, const unsigned *kept, int n, int nnz,
                                            const DmFastParams &P, int c0, int lane, bool wipe_after, unsigned &n_red)
{
    const unsigned nb = (unsigned)(P.bp.n_par * P.bp.n_perp);
    double *const Dn = P.Dn;
    const unsigned col0 = (unsigned)(c0 * P.bp.n_par);
#ifdef LYA_ABL_NO_T4
    if (n > 0) n = 0;
#endif
    for (int e0 = 0; e0 < n || (wipe_after && e0 == 0); e0 += FD_T4B) {
        double2 k01[FD_T4B], k23[FD_T4B];
        unsigned ro[FD_T4B];
#pragma unroll
        for (int k = 0; k < FD_T4B; ++k) {
            const int e = min(e0 + k, max(n - 1, 0));
            k01[k] = ws.u.b.kc01[e];
            k23[k] = ws.u.b.kc23[e];
            ro[k] = (kept[e] >> 16) * nb + col0;
        }
        const int m = min(FD_T4B, n - e0);
        const bool wipe = wipe_after && e0 + FD_T4B >= n;
#pragma unroll 1
        for (int t = lane; t < nnz; t += 32) {
            const unsigned slot = ws.u.b.nz[t];
            const double2 a = tb.H01[slot], b = tb.H23[slot];
            if (wipe) { tb.H01[slot] = make_double2(0.0, 0.0); tb.H23[slot] = make_double2(0.0, 0.0); }
#pragma unroll
            for (int k = 0; k < FD_T4B; ++k)
                if (k < m) dm_red(Dn + (ro[k] + slot), fma(k23[k].y, b.y, fma(k23[k].x, b.x, fma(k01[k].y, a.y, k01[k].x * a.x))));
        }
        if (lane == 0) n_red += (unsigned)(max(m, 0) * nnz);
    }
}

// table pool: lane 0 claims a free table (owner flag 0 -> 1), probing round-robin from the warp's own slot
template <int CLS>
__device__ __forceinline__ int dm_table_acquire(int *owner, int wid, int lane)
{
    int t = 0;
    if (lane == 0) {
        const int t0 = wid % FD_NTABLES;
        t = t0;
        while (atomicCAS(&owner[t], 0, 1) != 0) {
            t = (t + 1 == FD_NTABLES) ? 0 : t + 1;
            __nanosleep(64);
        }
        __threadfence_block();
    }
    return __shfl_sync(0xffffffffu, t, 0);
}
__device__ __forceinline__ void dm_table_release(int *owner, int t, int lane)
{
    __syncwarp();
    if (lane == 0) { __threadfence_block(); atomicExch(&owner[t], 0); }
}

template <bool POW2, bool CHECK, int CLS>
__global__ void __launch_bounds__(FD_THREADS, 1) k_dmat_fast(DmFastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int *owner = (int *)smem_raw;
    DmTable *tables = (DmTable *)(smem_raw + FD_POOL_HDR);
    DmFastWarp<CLS> &ws = ((DmFastWarp<CLS> *)(smem_raw + FD_POOL_HDR + sizeof(DmTable) * FD_NTABLES))[wid];
    const BinParams bp = P.bp;
    const unsigned npar = (unsigned)bp.n_par;
    const int n_slots = bp.n_par * LYA_NCOL;                  // real slots; slot n_slots is the garbage entry
    for (int t = threadIdx.x; t < FD_NTABLES * FD_SLOTS; t += FD_THREADS) {
        tables[t / FD_SLOTS].H01[t % FD_SLOTS] = make_double2(0.0, 0.0);
        tables[t / FD_SLOTS].H23[t % FD_SLOTS] = make_double2(0.0, 0.0);
    }
    if (threadIdx.x < FD_NTABLES) owner[threadIdx.x] = 0;
    if (lane < FD_PAD) { ws.qce[lane] = make_double2(LYA_CHI_SENTINEL, 0.0); ws.qeg[lane] = 0.0; }
    if (lane == 0) ws.nkept = 0u;
    __syncthreads();
    const double2 *qce = ws.qce + FD_PAD;
#ifdef LYA_ABL_NO_MASK
    const bool keep_none = true;
#else
    const bool keep_none = P.thr > 0xffffffffull;              // reject_fraction = 1
#endif
    const unsigned thr32 = (unsigned)P.thr;
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
            if (key >= 2 * bp.n_perp) continue;              // cannot happen in the fast ranges
            const unsigned lim = (unsigned)min(LYA_NCOL, bp.n_perp - c0);
            // lanes of a row step sit ds pixels of q apart; the class-0 range of the bucketed list holds only forest pairs
            // with ds == 1 (lya_pair_key), and a compile-time 1 folds the divisions by the stride out of the walk set-up
            const int ds = (CLS == 0) ? 1 : lya_pair_stride(bp, g, hq);
            __syncwarp();
            // ---- stage p (when it changes) and q: (chi, ea) pairs with 16-byte loads, eg, q's stage-4 keys ----
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
                if (!keep_none)
                    for (int t = lane; t < mq; t += 32) ws.u.a.qk[t] = lya_key_hi(P.seed, (unsigned long long)(hq.pix0 + t));
                if (lane < FD_PAD) {
                    const int j = FD_PAD + npad + lane;
                    ws.qce[j] = make_double2(LYA_CHI_SENTINEL, 0.0); ws.qeg[j] = 0.0;
                }
            }
            __syncwarp();
            // ---- windows (lanes over rows): the exact in-grid window [jlo, jhi) of q and the sign change jx;
            //      mask (same lanes): stage 4 over the window, pure integer; kept pairs (1 % at f = 0.99) are
            //      queued as (i, j) through a shared counter ----
            const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;
            const double Tchi = (s > 0.0) ? (bp.rperp_max / s) * (1.0 + 1e-12) + 1e-9 : 1e300;
            unsigned binned = 0;
            for (int ib = 0; ib < mp; ib += 32) {            // (warp-uniform trip counts: the warp must not stay split)
                const int i = ib + lane;
                if (i < mp) {
                    int jlo, jx, jhi;
                    lya_row_window_ilp<POW2, (FD_T < 128 ? 64 : 128)>(bp, g, qce, mq, ws.pce[i].x, R, Tchi, jlo, jx, jhi);
                    ws.jlo[i] = (unsigned char)jlo; ws.jx[i] = (unsigned char)jx; ws.jhi[i] = (unsigned char)jhi;
                    binned += (unsigned)(jhi - jlo);
                }
            }
            __syncwarp();
            if (!keep_none) {
                // Balanced scan: the in-window pairs of all rows form one list of M entries (row-major); lane l
                // takes entries [l K, (l + 1) K), K = ceil(M / 32).  pre[] (rows before i) is a warp scan with three
                // consecutive rows per lane; a lane finds its first row by binary search and then walks along,
                // stepping to the next non-empty row when its window ends.
                const int r3 = FD_RPL * lane;
                unsigned wrow[FD_RPL], incl = 0;
#pragma unroll
                for (int k = 0; k < FD_RPL; ++k) {
                    wrow[k] = (r3 + k < mp) ? (unsigned)ws.jhi[r3 + k] - ws.jlo[r3 + k] : 0u;
                    incl += wrow[k];
                }
                const unsigned own = incl;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const unsigned v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
                const unsigned M = __shfl_sync(0xffffffffu, incl, 31);
                unsigned run = incl - own;
#pragma unroll
                for (int k = 0; k < FD_RPL; ++k) {
                    if (r3 + k <= mp) ws.u.a.pre[r3 + k] = (unsigned short)run;
                    run += wrow[k];
                }
                for (int t = lane; t < mp; t += 32) ws.u.a.pk[t] = lya_key_lo(P.seed, (unsigned long long)(hp.pix0 + t));
                if (lane == 0) { ws.jlo[mp] = 0; ws.jhi[mp] = 0xff; }          // stop row: never left, never counted
                __syncwarp();
                const unsigned K = (M + 31u) >> 5;
                const unsigned first = min((unsigned)lane * K, M), last = min(first + K, M);
                int row = 0;
                {   // last row with pre[row] <= first  (pre is non-decreasing, pre[0] = 0)
                    int lo = 0, hi = mp;
                    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (ws.u.a.pre[mid] <= first) lo = mid; else hi = mid - 1; }
                    row = lo;
                }
                int j = (int)ws.jlo[row] + (int)(first - ws.u.a.pre[row]);
                int jend = (row >= mp) ? (1 << 30) : (int)ws.jhi[row];
                unsigned long long pki = ws.u.a.pk[min(row, FD_T - 1)];
                const unsigned n_it = __reduce_max_sync(0xffffffffu, last - first);
                unsigned long long qv = ws.u.a.qk[min(j, FD_T - 1)];
                for (unsigned t = 0; t < n_it; ++t) {
                    if (j >= jend) {                             // next non-empty row (the stop row ends the search)
                        do { ++row; } while (ws.jlo[row] == ws.jhi[row]);
                        j = ws.jlo[row]; jend = (row >= mp) ? (1 << 30) : (int)ws.jhi[row];
                        pki = ws.u.a.pk[min(row, FD_T - 1)];
                        qv = ws.u.a.qk[min(j, FD_T - 1)];
                    }
                    const unsigned long long qn = ws.u.a.qk[min(j + 1, FD_T - 1)];      // the row's next pixel, ahead of its use
                    const unsigned h = lya_pair_hash32(pki, qv);
                    qv = qn;
                    if ((first + t < last) & (h >= thr32)) {
                        const unsigned idx = atomicAdd(&ws.nkept, 1u);
                        if (idx < FD_KCAP) ws.kept[idx] = ((unsigned)row << 8) | (unsigned)j;
                    }
                    ++j;
                }
            }
            binned_total += binned;
            __syncwarp();
            const unsigned nk = ws.nkept;
            kept_total += (lane == 0) ? nk : 0u;
            // ---- pass C, first half: T1..T3 of the queued kept pairs (no H table needed yet).  Normally the
            //      queue holds every kept pair; with more than it holds (small reject fractions) the mask is
            //      redone row by row further down and the queue drained each time it fills ----
            const bool overflow = nk > FD_KCAP;
            const int n_q0 = overflow ? 0 : (int)nk;
            unsigned n_red32 = 0;
            for (int e0 = 0; e0 < n_q0; e0 += FD_KBATCH) {
                dm_drain_t123<POW2, CLS>(ws, ws.kept + e0, min(FD_KBATCH, n_q0 - e0), mp, P, g, hp.off, hq.off, lane, true, n_red32);
                __syncwarp();
            }
            // ---- pass A: H tables, in a table of the pool ----
            const int tix = dm_table_acquire<CLS>(owner, wid, lane);
            DmTable &tb = tables[tix];
            const unsigned h01 = (unsigned)__cvta_generic_to_shared(tb.H01);
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
#ifdef LYA_ABL_NO_WALK
                    continue;
#endif
                    dm_walk_any<POW2, CHECK>(ws, h01, r0 & ~1, r1 | 1, mq, sgn ? nlo : plo, sgn ? nhi : phi, ds, sgn, bp, g,
                                             (unsigned)c0, lim, npar, lane, evaluated, conflicts);
                }
            }
            __syncwarp();
            // ---- pass B: compact the non-zero entries (H_aa > 0 wherever a pair with weight fell) ----
            int nnz = 0;
            for (int t0 = 0; t0 < n_slots; t0 += 32) {
                const int t = t0 + lane;
                bool nzf = false;
                if (t < n_slots) nzf = tb.H01[t].x != 0.0;     // H_aa: a sum of products of non-negative ea, zero only where the other three are
                const unsigned bal = __ballot_sync(0xffffffffu, nzf);
                if (nzf) ws.u.b.nz[nnz + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)t;
                nnz += __popc(bal);
            }
            __syncwarp();
            // ---- pass C, second half: T4 (and, in the overflow case, the whole drain batch by batch) ----
            if (!overflow) {
                if (n_q0 <= FD_KBATCH) {                     // the coefficients of the only batch are still in place
                    dm_drain_t4<CLS>(ws, tb, ws.kept, n_q0, nnz, P, c0, lane, true, n_red32);
                } else {
                    for (int e0 = 0; e0 < n_q0; e0 += FD_KBATCH) {
                        const int nb_e = min(FD_KBATCH, n_q0 - e0);
                        dm_drain_t123<POW2, CLS>(ws, ws.kept + e0, nb_e, mp, P, g, hp.off, hq.off, lane, false, n_red32);
                        dm_drain_t4<CLS>(ws, tb, ws.kept + e0, nb_e, nnz, P, c0, lane, e0 + FD_KBATCH >= n_q0, n_red32);
                        __syncwarp();
                    }
                }
            } else {
                int si = 0, sj = (mp > 0) ? (int)ws.jlo[0] : 0;
                for (;;) {
                    int n_q = 0;
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
                    const bool done = si >= mp;
                    __syncwarp();
                    for (int e0 = 0; e0 < n_q || e0 == 0; e0 += FD_KBATCH) {
                        const int nb_e = max(min(FD_KBATCH, n_q - e0), 0);
                        dm_drain_t123<POW2, CLS>(ws, ws.kept + e0, nb_e, mp, P, g, hp.off, hq.off, lane, true, n_red32);
                        dm_drain_t4<CLS>(ws, tb, ws.kept + e0, nb_e, nnz, P, c0, lane, done && e0 + FD_KBATCH >= n_q, n_red32);
                        __syncwarp();
                    }
                    if (done) break;
                }
            }
            n_red += n_red32;
            // the garbage entry collects every out-of-grid product: clear it too, then hand the table back
            if (lane == 0) { tb.H01[n_slots] = make_double2(0.0, 0.0); tb.H23[n_slots] = make_double2(0.0, 0.0); ws.nkept = 0u; }
            dm_table_release(owner, tix, lane);
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

#undef FD_WARPS
#undef FD_THREADS
#undef FD_T
#undef FD_TP
#undef FD_TQ
#undef FD_KCAP
#undef FD_RPL
#undef FD_NTABLES
