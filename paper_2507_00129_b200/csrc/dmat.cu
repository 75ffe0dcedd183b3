// dmat.cu -- stages 3+4 (lya_dmat): distortion matrix of eqs. 2.6-2.7
// with the seeded pixel-pair keep mask.
//
//   D_AB = W_A^-1 sum_{(i,j) in A, kept} w_i w_j sum_{(i',j') in B} eta_ii' eta_jj'
//   eta_ii' = delta^K_ii' - a_i' - u_i g_i'   (identity minus rank 2; eq. 2.7 with
//   a = w / sum w,  u = L - Lbar (w-weighted mean, reading R-10),  g = w u / sum w u^2)
//
// The inner double sum collapses (the CPU oracle does NOT use this; it evaluates the
// naive quadruple sum with explicit eta matrices).  For a kept pair (i,j) in bin A,
// om = w_i w_j, and H_xy[B] = sum_{(i',j') in B} x_i' y_j' over the forest pair:
//   Dn[A][A]            += om                                            (T1)
//   Dn[A][bin(i ,j')]   -= om (a_j' + u_j g_j')      for every j' in q   (T2)
//   Dn[A][bin(i',j )]   -= om (a_i' + u_i g_i')      for every i' in p   (T3)
//   Dn[A][B]            += om (H_aa + u_j H_ag + u_i H_ga + u_i u_j H_gg)[B]   (T4)
// so a forest pair costs one O(n_p n_q) pass for the four H tables and then
// ~(n_p + n_q + |support|) scatter-adds per KEPT pair.  The scatter is a sparse
// rank-4 update (about 14 kept pairs x 116 bins per forest pair at f = 0.99): not a
// dense GEMM, so no tensor cores.
//
// Two kernels, one warp per forest pair in both, every update one red.global.add.f64 into the
// L2-resident Dn (kept in TRANSPOSED bin order b_perp * n_par + b_par; k_dmat_normalise permutes):
//   k_dmat_fast  (below, second half of the file) for the pairs of the bucketed list: H tables by the
//                xi kernel's diagonal walk with entries held in registers, mask hashed on the fly,
//                compacted drain -- see its header;
//   k_dmat       generic: forests of any length in 128-pixel tiles, any column span (chunks of LC
//                columns), any pixel spacing; H tables with CAS shared atomics (pass 1a), mask and
//                drain per tile pair (pass 1b), T2/T3 read the whole forests from global memory.
// lya_pairs_subsample (forest-pair subsampling) lives here too: it shares the mask.
#include <stdlib.h>
#include "lya_internal.cuh"

namespace {

constexpr int DM_WARPS = 4;
constexpr int DM_THREADS = DM_WARPS * 32;
constexpr int DTILE = 128;               // max pixels per forest handled by this kernel
constexpr int DQPAD = 4;
constexpr int H_SLOTS = 512;             // local (b_par, column) slots per H table
constexpr int KEPT_CAP = 256;
constexpr int DCHUNK = 8;

// ---- stage 4: the keep mask (integer only) -------------------------
__device__ __forceinline__ unsigned long long mix64(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__device__ __forceinline__ unsigned long long key_lo(unsigned long long seed, unsigned long long id)
{
    return mix64(seed + id * 0x9E3779B97F4A7C15ULL);
}
__device__ __forceinline__ unsigned long long key_hi(unsigned long long seed, unsigned long long id)
{
    return mix64((seed ^ 0xD1B54A32D192ED03ULL) + id * 0x9E3779B97F4A7C15ULL);
}
__device__ __forceinline__ bool keep_pair(unsigned long long klo, unsigned long long khi, unsigned long long thr)
{
    unsigned long long x = klo + khi;
    x ^= x >> 32;
    x *= 0xD6E8FEB86659FD93ULL;
    return (x >> 32) >= thr;
}

struct DmParams {
    const int64_t *pix_off;
    const double *chi, *w, *loglam;
    const double *ux, *uy, *uz;
    const double *f_invS, *f_lbar, *f_invV;      // per forest
    const int32_t *pq;
    int64_t n_pairs, n_forest;
    BinParams bp;
    unsigned long long seed, thr;
    double *Dn, *Wd;
    unsigned long long *counters;   // [0] next chunk, [1] visited, [2] evaluated, [3] error, [5] kept, [6] binned
    int LC;                         // columns per local table
};

// per-forest scalars of eq. 2.7: 1/sum w, Lbar, 1/sum w (L-Lbar)^2 (NaN when degenerate)
__global__ void k_forest_scalars(const int64_t *pix_off, const double *w, const double *loglam, int64_t n_forest,
                                 double *invS, double *lbar, double *invV)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= n_forest) return;
    int64_t a = pix_off[p], b = pix_off[p + 1];
    double sw = 0.0, swl = 0.0;
    for (int64_t k = a; k < b; ++k) { sw += w[k]; swl += w[k] * loglam[k]; }
    double lb = (sw > 0.0) ? swl / sw : 0.0;
    double v = 0.0;
    for (int64_t k = a; k < b; ++k) { double u = loglam[k] - lb; v += w[k] * u * u; }
    bool ok = (sw > 0.0) && (v > 0.0);
    invS[p] = ok ? 1.0 / sw : nan("");
    lbar[p] = lb;
    invV[p] = ok ? 1.0 / v : nan("");
}

struct DmWarpSmem {
    double pc[DTILE], pw[DTILE], pu[DTILE];
    unsigned long long pk[DTILE];
    double qc[DTILE + 2 * DQPAD], qw[DTILE + 2 * DQPAD], qu[DTILE + 2 * DQPAD];
    unsigned long long qk[DTILE];
    double H[4][H_SLOTS];
    unsigned kept[KEPT_CAP];        // (i << 20) | (j << 12) | bin
    unsigned short nz[H_SLOTS];     // non-zero slots of the H tables of the current column chunk
};

__device__ __forceinline__ void red_add(double *addr, double v) { atomicAdd(addr, v); }

// Drain the kept-pair queue of one staged tile pair: T1..T3 (first column chunk only) and T4 (this
// chunk's columns).  T2 / T3 run over the WHOLE forests q / p, read from global memory (forests can
// be longer than a tile); op, oq = offsets of the forests, np, nq = their lengths.
template <bool POW2>
__device__ void drain_kept(DmWarpSmem &ws, int n_kept, const DmParams &P, const PairBin &g,
                           int64_t op, int np, double lbp, double invSp, double invVp,
                           int64_t oq, int nq, double lbq, double invSq, double invVq,
                           int c0, int ncol, int nnz, bool first_chunk, int lane)
{
    const BinParams &bp = P.bp;
    const int nb = bp.n_par * bp.n_perp;
    const double *qc = ws.qc + DQPAD, *qw = ws.qw + DQPAD, *qu = ws.qu + DQPAD;
    for (int e = 0; first_chunk && e < n_kept; ++e) {
        const unsigned rec = ws.kept[e];
        const int i = rec >> 20, j = (rec >> 12) & 0xff, A = rec & 0xfff;
        const double om = ws.pw[i] * qw[j];
        const double ui = ws.pu[i], uj = qu[j];
        const int At = lya_bin_tr(bp, A);                                  // Dn, Wd are accumulated in transposed bin order
        double *row = P.Dn + (size_t)At * nb;
        if (lane == 0) { red_add(row + At, om); red_add(P.Wd + At, om); }
        for (int j2 = lane; j2 < nq; j2 += 32) {                           // T2
            int B = lya_pix_bin_t<POW2>(bp, g, ws.pc[i], P.chi[oq + j2]);
            if (B >= 0) {
                const double w2 = P.w[oq + j2], u2 = P.loglam[oq + j2] - lbq;
                red_add(row + B, -om * (w2 * invSq + uj * (w2 * u2 * invVq)));
            }
        }
        for (int i2 = lane; i2 < np; i2 += 32) {                           // T3
            int B = lya_pix_bin_t<POW2>(bp, g, P.chi[op + i2], qc[j]);
            if (B >= 0) {
                const double w2 = P.w[op + i2], u2 = P.loglam[op + i2] - lbp;
                red_add(row + B, -om * (w2 * invSp + ui * (w2 * u2 * invVp)));
            }
        }
    }
    // T4: lanes over the non-zero table entries of this column chunk, inner loop over the kept pairs
    for (int t = lane; t < nnz; t += 32) {
        const int slot = ws.nz[t];
        const int bx = slot / ncol, lc = slot - bx * ncol;
        double *colB = P.Dn + ((c0 + lc) * bp.n_par + bx);
        const double h0 = ws.H[0][slot], h1 = ws.H[1][slot], h2 = ws.H[2][slot], h3 = ws.H[3][slot];
        for (int e = 0; e < n_kept; ++e) {
            const unsigned rec = ws.kept[e];
            const int i = rec >> 20, j = (rec >> 12) & 0xff, A = rec & 0xfff;
            const double om = ws.pw[i] * qw[j], ui = ws.pu[i], uj = qu[j];
            red_add(colB + (size_t)lya_bin_tr(bp, A) * nb, om * ((h0 + uj * h1) + ui * (h2 + uj * h3)));
        }
    }
}

template <bool POW2>
__global__ void __launch_bounds__(DM_THREADS) k_dmat(DmParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DmWarpSmem &ws = ((DmWarpSmem *)smem_raw)[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const BinParams bp = P.bp;
    const int LC = P.LC;
    unsigned long long visited = 0, evaluated = 0, kept_total = 0, binned = 0;
    const int64_t n_chunks = (P.n_pairs + DCHUNK - 1) / DCHUNK;
    int cur_p = -1, cur_ip0 = -1, scal_p = -1;
    double invSp = 0, invVp = 0, lbp = 0;
    const double *qc = ws.qc + DQPAD, *qw = ws.qw + DQPAD, *qu = ws.qu + DQPAD;

    for (;;) {
        unsigned long long chunk = 0;
        if (lane == 0) chunk = atomicAdd(&P.counters[0], 1ull);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if ((int64_t)chunk >= n_chunks) break;
        const int64_t k0 = (int64_t)chunk * DCHUNK, k1 = min(k0 + DCHUNK, P.n_pairs);
        for (int64_t k = k0; k < k1; ++k) {
            const int p = P.pq[2 * k], q = P.pq[2 * k + 1];
            if ((unsigned)p >= (unsigned)P.n_forest || (unsigned)q >= (unsigned)P.n_forest) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_BAD_PAIR);
                continue;
            }
            const int64_t op = P.pix_off[p], oq = P.pix_off[q];
            const int np = (int)(P.pix_off[p + 1] - op), nq = (int)(P.pix_off[q + 1] - oq);
            if (np == 0 || nq == 0) continue;
            const double invSq = P.f_invS[q], invVq = P.f_invV[q], lbq = P.f_lbar[q];
            if (p != scal_p) { invSp = P.f_invS[p]; invVp = P.f_invV[p]; lbp = P.f_lbar[p]; scal_p = p; }
            if (isnan(invSp) || isnan(invVp) || isnan(invSq) || isnan(invVq)) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_DEGENERATE);
                continue;
            }
            visited += (unsigned long long)np * nq;
            double s, c;
            lya_pair_sc(P.ux[p], P.uy[p], P.uz[p], P.ux[q], P.uy[q], P.uz[q], s, c);
            const PairBin g = lya_make_pairbin(bp, s, c);
            // r_perp column range of this forest pair: r_perp is increasing in both pixels
            int c_first, c_last;
            {
                double t0 = __dmul_rn(__dadd_rn(P.chi[op], P.chi[oq]), g.s);
                double t1 = __dmul_rn(__dadd_rn(P.chi[op + np - 1], P.chi[oq + nq - 1]), g.s);
                if (!(t0 < bp.rperp_max)) continue;                        // nothing in the grid
                c_first = min((int)lya_floor_u32(__dmul_rn(t0, bp.inv_perp)), bp.n_perp - 1);
                c_last = (t1 < bp.rperp_max) ? min((int)lya_floor_u32(__dmul_rn(t1, bp.inv_perp)), bp.n_perp - 1)
                                             : bp.n_perp - 1;
            }
            // stage one DTILE-pixel tile of p / q (forests of any length are walked tile by tile)
            auto stage_p = [&](int ip0, int mp) {
                if (p == cur_p && ip0 == cur_ip0) return;
                __syncwarp();
                for (int t = lane; t < mp; t += 32) {
                    ws.pc[t] = P.chi[op + ip0 + t];
                    ws.pw[t] = P.w[op + ip0 + t];
                    ws.pu[t] = P.loglam[op + ip0 + t] - lbp;
                    ws.pk[t] = key_lo(P.seed, (unsigned long long)(op + ip0 + t));
                }
                cur_p = p; cur_ip0 = ip0;
                __syncwarp();
            };
            auto stage_q = [&](int jq0, int mq) {
                __syncwarp();
                for (int t = lane; t < mq + 2 * DQPAD; t += 32) {
                    int j = t - DQPAD;
                    bool in = (j >= 0) && (j < mq);
                    ws.qc[t] = in ? P.chi[oq + jq0 + j] : LYA_CHI_SENTINEL;
                    ws.qw[t] = in ? P.w[oq + jq0 + j] : 0.0;
                    ws.qu[t] = in ? P.loglam[oq + jq0 + j] - lbq : 0.0;
                    if (in) ws.qk[j] = key_hi(P.seed, (unsigned long long)(oq + jq0 + j));
                }
                __syncwarp();
            };
            for (int c0 = c_first; c0 <= c_last; c0 += LC) {
                const int ncol = min(LC, c_last - c0 + 1);
                const bool first_chunk = (c0 == c_first);
                const int n_slots = bp.n_par * ncol;
                __syncwarp();
                for (int t = lane; t < n_slots; t += 32) { ws.H[0][t] = 0.0; ws.H[1][t] = 0.0; ws.H[2][t] = 0.0; ws.H[3][t] = 0.0; }
                __syncwarp();
                // ---- pass 1a: H tables over every tile pair; lanes own diagonals d = j - i, register run-length ----
                for (int ip0 = 0; ip0 < np; ip0 += DTILE) {
                    const int mp = min(DTILE, np - ip0);
                    stage_p(ip0, mp);
                    for (int jq0 = 0; jq0 < nq; jq0 += DTILE) {
                        const int mq = min(DTILE, nq - jq0);
                        stage_q(jq0, mq);
                        for (int d0 = -(mp - 1); d0 <= mq - 1; d0 += 32) {
                            const int d = d0 + lane;
                            const int i_begin = max(0, -min(mq - 1, d0 + 31));
                            const int i_end = min(mp, mq - d0);
                            int cur = -1;
                            double h0 = 0, h1 = 0, h2 = 0, h3 = 0;
                            evaluated += (unsigned long long)(i_end - i_begin);
                            for (int i = i_begin; i < i_end; ++i) {
                                int j = min(max(i + d, -DQPAD), mq + DQPAD - 1);
                                int bin = lya_pix_bin<POW2>(bp, g, ws.pc[i], qc[j]);
                                int slot = -1;
                                if (bin >= 0) {
                                    int bx = bin / bp.n_perp, by = bin - bx * bp.n_perp;
                                    if (by >= c0 && by < c0 + ncol) slot = bx * ncol + (by - c0);
                                }
                                if (slot != cur) {
                                    if (cur >= 0) {
                                        atomicAdd(&ws.H[0][cur], h0); atomicAdd(&ws.H[1][cur], h1);
                                        atomicAdd(&ws.H[2][cur], h2); atomicAdd(&ws.H[3][cur], h3);
                                    }
                                    cur = slot; h0 = h1 = h2 = h3 = 0.0;
                                }
                                if (slot >= 0) {
                                    double ai = ws.pw[i] * invSp, gi = ws.pw[i] * ws.pu[i] * invVp;
                                    double aj = qw[j] * invSq, gj = qw[j] * qu[j] * invVq;
                                    h0 = fma(ai, aj, h0); h1 = fma(ai, gj, h1);
                                    h2 = fma(gi, aj, h2); h3 = fma(gi, gj, h3);
                                }
                            }
                            if (cur >= 0) {
                                atomicAdd(&ws.H[0][cur], h0); atomicAdd(&ws.H[1][cur], h1);
                                atomicAdd(&ws.H[2][cur], h2); atomicAdd(&ws.H[3][cur], h3);
                            }
                        }
                    }
                }
                __syncwarp();
                int nnz = 0;                                               // compact the non-zero entries once per chunk
                for (int t0 = 0; t0 < n_slots; t0 += 32) {
                    const int t = t0 + lane;
                    const bool nzf = t < n_slots && (ws.H[0][t] != 0.0 || ws.H[1][t] != 0.0 || ws.H[2][t] != 0.0 || ws.H[3][t] != 0.0);
                    const unsigned bal = __ballot_sync(0xffffffffu, nzf);
                    if (nzf) ws.nz[nnz + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)t;
                    nnz += __popc(bal);
                }
                __syncwarp();
                // ---- pass 1b: mask every in-grid pair of every tile pair, queue the kept ones, drain ----
                for (int ip0 = 0; ip0 < np; ip0 += DTILE) {
                    const int mp = min(DTILE, np - ip0);
                    stage_p(ip0, mp);
                    for (int jq0 = 0; jq0 < nq; jq0 += DTILE) {
                        const int mq = min(DTILE, nq - jq0);
                        stage_q(jq0, mq);
                        int n_q = 0;
                        for (int i = 0; i < mp; ++i) {
                            const double pci = ws.pc[i];
                            const unsigned long long ki = ws.pk[i];
                            for (int j0 = 0; j0 < mq; j0 += 32) {
                                const int j = j0 + lane;
                                int bin = -1;
                                if (j < mq) bin = lya_pix_bin<POW2>(bp, g, pci, qc[j]);
                                bool kp = (bin >= 0) && keep_pair(ki, ws.qk[min(j, mq - 1)], P.thr);
                                if (first_chunk) {
                                    binned += (bin >= 0);
                                    kept_total += kp;
                                }
                                unsigned bal = __ballot_sync(0xffffffffu, kp);
                                if (bal) {
                                    if (n_q + __popc(bal) > KEPT_CAP) {
                                        __syncwarp();
                                        drain_kept<POW2>(ws, n_q, P, g, op, np, lbp, invSp, invVp, oq, nq, lbq, invSq, invVq, c0, ncol, nnz, first_chunk, lane);
                                        __syncwarp();
                                        n_q = 0;
                                    }
                                    if (kp) ws.kept[n_q + __popc(bal & ((1u << lane) - 1u))] = ((unsigned)i << 20) | ((unsigned)j << 12) | (unsigned)bin;
                                    n_q += __popc(bal);
                                }
                            }
                        }
                        __syncwarp();
                        drain_kept<POW2>(ws, n_q, P, g, op, np, lbp, invSp, invVp, oq, nq, lbq, invSq, invVq, c0, ncol, nnz, first_chunk, lane);
                        __syncwarp();
                    }
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
        kept_total += __shfl_xor_sync(0xffffffffu, kept_total, o);
        binned += __shfl_xor_sync(0xffffffffu, binned, o);
    }
    if (lane == 0) {
        atomicAdd(&P.counters[1], visited);
        atomicAdd(&P.counters[2], evaluated);
        atomicAdd(&P.counters[5], kept_total);
        atomicAdd(&P.counters[6], binned);
    }
}

// ======================= fast kernel ======================================
// One warp per forest pair of the bucket-sorted list, forests staged from the padded catalogue.
//  pass A  diagonal walk (the xi kernel's traversal): the four H tables of the pair, each lane
//          holding the table entry of its current run in registers (predicated release/acquire, no
//          atomics: the walk is done once per side of chi_i = chi_j, so entries have one holder);
//          every in-grid pair is hashed on the fly (stage 4) and the kept ones are queued;
//  pass B  the non-zero table entries are compacted into a list;
//  pass C  the kept pairs are drained: T1..T3 per kept pair, T4 with lanes over the table entries and
//          an inner loop over the kept pairs (the entry stays in registers); every update is one
//          red.global.add.f64 into the L2-resident Dn.
constexpr int FD_WARPS = 15;                 // one CTA per SM (shared memory: 15.1 KB per warp)
constexpr int FD_THREADS = FD_WARPS * 32;
constexpr int FD_T = LYA_FAST_TILE;
constexpr int FD_ROWS = 16;
constexpr int FD_TP = ((FD_T + FD_ROWS - 1) / FD_ROWS) * FD_ROWS + 2;
constexpr int FD_PAD = 2;
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
    unsigned long long *counters;   // [4] next chunk, [2] evaluated, [3] error, [5] kept, [6] binned, [7] scatter-adds
};

struct DmKeysA { unsigned long long pk[FD_T], qk[FD_T]; };                 // pass A: stage-4 keys of the pixels
struct DmDrainBC {                                                            // passes B and C
    double2 kc01[FD_KBATCH], kc23[FD_KBATCH];    // per kept pair of a batch: om (1, u_j), om (u_i, u_i u_j)
    unsigned short nz[FD_SLOTS];                 // non-zero slots
};
struct __align__(16) DmFastWarp {
    double2 H01[FD_SLOTS], H23[FD_SLOTS];    // (H_aa, H_ag), (H_ga, H_gg) per slot = col_rel * (n_par + 1) + row
    double pc[FD_TP], pea[FD_TP], peg[FD_TP];            // (w and u of the kept pairs are read from HBM/L2 in the drain)
    double qc[FD_T + 2 * FD_PAD], qea[FD_T + 2 * FD_PAD], qeg[FD_T + 2 * FD_PAD];
    union { DmKeysA a; DmDrainBC b; } u;     // the keys are dead once pass A is done (shared memory buys occupancy)
    unsigned kept[FD_KCAP];                  // (i << 20) | (j << 12) | A
    unsigned char jlo[FD_T], jx[FD_T], jhi[FD_T];
    unsigned nkept, pad_[3];
};

__device__ __forceinline__ void dsts_v2_if(bool p, unsigned addr, double x, double y)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %0, 0;\n @q st.shared.v2.f64 [%1], {%2, %3};\n}"
                 :: "r"((unsigned)p), "r"(addr), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void dlds_v2_if(bool p, unsigned addr, double &x, double &y)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %2, 0;\n @q ld.shared.v2.f64 {%0, %1}, [%3];\n}"
                 : "+d"(x), "+d"(y) : "r"((unsigned)p), "r"(addr) : "memory");
}

// byte offset (16 * slot) of a pixel pair in the H tables and whether it is a pair of THIS walk
// (inside the grid and on the walk's side of chi_i = chi_j: sgn = 0 for chi_i >= chi_j, -1 otherwise);
// A = its bin.  Pairs outside get the garbage row / column.
template <bool POW2>
__device__ __forceinline__ unsigned dm_key(const BinParams &bp, const PairBin &g, double chi_i, double chi_j, unsigned c0,
                                           unsigned np1, int sgn, bool &valid, unsigned &A)
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
    const bool side = ((__double2hiint(d) ^ sgn) >= 0);
    valid = side & (bx < (unsigned)bp.n_par) & (by < (unsigned)bp.n_perp);
    A = by * (unsigned)bp.n_par + bx;                   // transposed bin order (see lya_pix_bin_t)
    bx = valid ? bx : np1 - 1u;                          // everything else -> the garbage entry (0, n_par)
    const unsigned col = valid ? by - c0 : 0u;
    return (col * np1 + bx) * 16u;
}

// stage-4 keep mask on precomputed pixel keys (same integer function as keep_pair above)
__device__ __forceinline__ bool dm_keep(unsigned long long klo, unsigned long long khi, unsigned long long thr)
{
    return keep_pair(klo, khi, thr);
}

// pass A over rows [r0, r1] (a multiple of D rows; rows >= len are sentinels) and diagonals [dlo, dhi].
// Same scheme as k_xi_fast: a lane holds the H entry of its current run in registers (predicated
// release / acquire around a warp barrier); the keys, mask and queueing of row i+1 are computed
// between the acquire of row i and the FMAs that need it.
template <int D, bool POW2>
__device__ __forceinline__ void dm_walk(DmFastWarp &ws, unsigned h01, unsigned h23, int r0, int r1, int mq, int dlo, int dhi,
                                        int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned np1,
                                        unsigned long long thr, int lane, unsigned &binned, unsigned &kept_n,
                                        unsigned long long &evaluated)
{
    const double *qc = ws.qc + FD_PAD, *qea = ws.qea + FD_PAD, *qeg = ws.qeg + FD_PAD;
    const unsigned garbage = (np1 - 1u) * 16u;
    for (int d0 = dlo; d0 <= dhi; d0 += 32 * D) {
        const int dl = d0 + lane * D;
        unsigned cur[D], key[D];
        double h0[D], h1[D], h2[D], h3[D], fa[D], fg[D];
        double wc[D], wa[D], wg[D];                         // sliding window over q: chi, ea, eg
        double pa_c, pg_c;
#pragma unroll
        for (int k = 0; k < D; ++k) { cur[k] = garbage; h0[k] = 0.0; h1[k] = 0.0; h2[k] = 0.0; h3[k] = 0.0; }
        // keys, mask and queueing of one row (i, window slot of diagonal k = (k + u) % D)
        auto row_keys = [&](int i, int u, bool live, unsigned *key_o, double *fa_o, double *fg_o) {
            const double pci = ws.pc[i];
            const unsigned long long pki = ws.u.a.pk[min(i, FD_T - 1)];
#pragma unroll
            for (int k = 0; k < D; ++k) {
                const int sl = (k + u) % D;
                bool valid; unsigned A;
                key_o[k] = dm_key<POW2>(bp, g, pci, wc[sl], c0, np1, sgn, valid, A);
                fa_o[k] = wa[sl]; fg_o[k] = wg[sl];
                valid = valid && live;
                const int j = i + dl + k;
                const bool kp = valid && keep_pair(pki, ws.u.a.qk[min(max(j, 0), FD_T - 1)], thr);
                binned += valid ? 1u : 0u;
                if (kp) {                                    // ~1 % of the pairs at f = 0.99
                    const unsigned idx = atomicAdd(&ws.nkept, 1u);
                    if (idx < FD_KCAP) ws.kept[idx] = ((unsigned)i << 20) | ((unsigned)j << 12) | A;
                    kept_n += 1u;
                }
            }
        };
#pragma unroll
        for (int k = 0; k < D; ++k) {
            const int j = min(max(r0 + dl + k, -FD_PAD), mq + FD_PAD - 1);
            wc[k] = qc[j]; wa[k] = qea[j]; wg[k] = qeg[j];
        }
        row_keys(r0, 0, true, key, fa, fg);
        pa_c = ws.pea[r0]; pg_c = ws.peg[r0];
        evaluated += (unsigned long long)(r1 - r0 + 1) * D;
        for (int ib = r0; ib <= r1; ib += D) {
#pragma unroll
            for (int u = 0; u < D; ++u) {
                const int i = ib + u;
                bool ch[D];
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    ch[k] = key[k] != cur[k];
                    dsts_v2_if(ch[k], h01 + cur[k], h0[k], h1[k]);                      // release
                    dsts_v2_if(ch[k], h23 + cur[k], h2[k], h3[k]);
                }
                __syncwarp();
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    dlds_v2_if(ch[k], h01 + key[k], h0[k], h1[k]);                      // acquire
                    dlds_v2_if(ch[k], h23 + key[k], h2[k], h3[k]);
                    cur[k] = key[k];
                }
                // row i + 1: its new q pixel replaces q[i + dl] in window slot u
                unsigned key_n[D];
                double fa_n[D], fg_n[D];
                {
                    const int j = min(max(i + dl + D, -FD_PAD), mq + FD_PAD - 1);
                    wc[u] = qc[j]; wa[u] = qea[j]; wg[u] = qeg[j];
                    row_keys(i + 1, u + 1, i + 1 <= r1, key_n, fa_n, fg_n);
                }
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    h0[k] = fma(pa_c, fa[k], h0[k]); h1[k] = fma(pa_c, fg[k], h1[k]);
                    h2[k] = fma(pg_c, fa[k], h2[k]); h3[k] = fma(pg_c, fg[k], h3[k]);
                    fa[k] = fa_n[k]; fg[k] = fg_n[k]; key[k] = key_n[k];
                }
                pa_c = ws.pea[i + 1]; pg_c = ws.peg[i + 1];
            }
        }
#pragma unroll
        for (int k = 0; k < D; ++k) {
            dsts_v2_if(true, h01 + cur[k], h0[k], h1[k]);
            dsts_v2_if(true, h23 + cur[k], h2[k], h3[k]);
        }
        __syncwarp();
    }
}

template <bool POW2>
__device__ __forceinline__ void dm_walk_any(DmFastWarp &ws, unsigned h01, unsigned h23, int r0, int r1, int mq, int dlo, int dhi,
                                            int sgn, const BinParams &bp, const PairBin &g, unsigned c0, unsigned np1,
                                            unsigned long long thr, int lane, unsigned &binned, unsigned &kept_n,
                                            unsigned long long &evaluated)
{
    if (dhi < dlo) return;
    const int nd = dhi - dlo + 1;
    if (nd <= 32) dm_walk<1, POW2>(ws, h01, h23, r0, r1, mq, dlo, dhi, sgn, bp, g, c0, np1, thr, lane, binned, kept_n, evaluated);
    else dm_walk<2, POW2>(ws, h01, h23, r0, r1, mq, dlo, dhi, sgn, bp, g, c0, np1, thr, lane, binned, kept_n, evaluated);
}

// pass C: drain n queued kept pairs.
template <bool POW2>
__device__ __forceinline__ void dm_drain_batch(DmFastWarp &ws, const unsigned *kept, int n, int nnz, int mp, int mq, const DmFastParams &P,
                                         const PairBin &g, int c0, long long offp, long long offq, int lane,
                                         unsigned long long &n_red)
{
    const BinParams &bp = P.bp;
    const int nb = bp.n_par * bp.n_perp, np1 = bp.n_par + 1;
    const double *qc = ws.qc + FD_PAD, *qea = ws.qea + FD_PAD, *qeg = ws.qeg + FD_PAD;
    // coefficients of every kept pair (lanes over kept pairs) and T1: Dn[A][A] += om, Wd[A] += om
    for (int e = lane; e < n; e += 32) {
        const unsigned rec = kept[e];
        const int i = rec >> 20, j = (rec >> 12) & 0xff, A = rec & 0xfff;
        const double om = P.prep.w[offp + i] * P.prep.w[offq + j], ui = P.prep.u[offp + i], uj = P.prep.u[offq + j];
        const double omi = om * ui;
        ws.u.b.kc01[e] = make_double2(om, om * uj);
        ws.u.b.kc23[e] = make_double2(omi, omi * uj);
        atomicAdd(P.Dn + (size_t)A * nb + A, om);
        atomicAdd(P.Wd + A, om);
        n_red += 2;
    }
    __syncwarp();
    // T2: -(om ea_j' + om u_j eg_j') over row i's window;  T3: -(om ea_i' + om u_i eg_i') over p
    for (int e = 0; e < n; ++e) {
        const unsigned rec = kept[e];
        const int i = rec >> 20, j = (rec >> 12) & 0xff, A = rec & 0xfff;
        const double2 c01 = ws.u.b.kc01[e], c23 = ws.u.b.kc23[e], geo = make_double2(ws.pc[i], qc[j]);
        double *row = P.Dn + (size_t)A * nb;
        for (int j2 = ws.jlo[i] + lane; j2 < ws.jhi[i]; j2 += 32) {
            const int B = lya_pix_bin_t<POW2>(bp, g, geo.x, qc[j2]);
            if (B >= 0) { atomicAdd(row + B, -fma(c01.y, qeg[j2], c01.x * qea[j2])); n_red += 1; }
        }
        for (int i2 = lane; i2 < mp; i2 += 32) {
            const int B = lya_pix_bin_t<POW2>(bp, g, ws.pc[i2], geo.y);
            if (B >= 0) { atomicAdd(row + B, -fma(c23.x, ws.peg[i2], c01.x * ws.pea[i2])); n_red += 1; }
        }
    }
    // T4: lanes over the non-zero table entries, inner loop over the kept pairs
    for (int t = lane; t < nnz; t += 32) {
        const int slot = ws.u.b.nz[t];
        const int cr = slot / np1, bx = slot - cr * np1;
        double *colB = P.Dn + ((c0 + cr) * bp.n_par + bx);
        const double2 a = ws.H01[slot], b = ws.H23[slot];
#pragma unroll 2
        for (int e = 0; e < n; ++e) {
            const int A = kept[e] & 0xfff;
            const double2 c01 = ws.u.b.kc01[e], c23 = ws.u.b.kc23[e];
            const double v = fma(c23.y, b.y, fma(c23.x, b.x, fma(c01.y, a.y, c01.x * a.x)));
            atomicAdd(colB + (size_t)A * nb, v);
        }
        n_red += (unsigned long long)n;
    }
}

template <bool POW2>
__device__ __forceinline__ void dm_drain(DmFastWarp &ws, int n, int nnz, int mp, int mq, const DmFastParams &P,
                                         const PairBin &g, int c0, long long offp, long long offq, int lane,
                                         unsigned long long &n_red)
{
    for (int e0 = 0; e0 < n; e0 += FD_KBATCH) {
        dm_drain_batch<POW2>(ws, ws.kept + e0, min(FD_KBATCH, n - e0), nnz, mp, mq, P, g, c0, offp, offq, lane, n_red);
        __syncwarp();
    }
}

template <bool POW2>
__global__ void __launch_bounds__(FD_THREADS, 1) k_dmat_fast(DmFastParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    DmFastWarp &ws = ((DmFastWarp *)smem_raw)[wid];
    const BinParams bp = P.bp;
    const unsigned np1 = (unsigned)bp.n_par + 1u;
    const int n_slots = (int)np1 * LYA_NCOL;
    for (int t = lane; t < FD_SLOTS; t += 32) { ws.H01[t] = make_double2(0.0, 0.0); ws.H23[t] = make_double2(0.0, 0.0); }
    if (lane < FD_PAD) { ws.qc[lane] = LYA_CHI_SENTINEL; ws.qea[lane] = 0.0; ws.qeg[lane] = 0.0; }
    if (lane == 0) ws.nkept = 0u;
    __syncwarp();
    const double *qc = ws.qc + FD_PAD;
    const unsigned h01 = (unsigned)__cvta_generic_to_shared(ws.H01), h23 = (unsigned)__cvta_generic_to_shared(ws.H23);
    unsigned long long evaluated = 0, kept_total = 0, binned_total = 0, n_red = 0;
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
            __syncwarp();
            if (p != cur_p) {
                const double2 *s0 = (const double2 *)(P.prep.chi + hp.off), *s3 = (const double2 *)(P.prep.ea + hp.off),
                              *s4 = (const double2 *)(P.prep.eg + hp.off);
                for (int t = lane; 2 * t < mp; t += 32) {
                    ((double2 *)ws.pc)[t] = s0[t]; ((double2 *)ws.pea)[t] = s3[t]; ((double2 *)ws.peg)[t] = s4[t];
                }
                __syncwarp();
                for (int t = mp + lane; t < FD_TP; t += 32) {            // sentinel rows (!= q's sentinel: r_par never 0)
                    ws.pc[t] = 2.0 * LYA_CHI_SENTINEL; ws.pea[t] = 0.0; ws.peg[t] = 0.0;
                }
                cur_p = p;
            }
            {
                const double2 *s0 = (const double2 *)(P.prep.chi + hq.off), *s3 = (const double2 *)(P.prep.ea + hq.off),
                              *s4 = (const double2 *)(P.prep.eg + hq.off);
                const int npad2 = (mq + 1) >> 1;
                for (int t = lane; t < npad2; t += 32) {
                    ((double2 *)qc)[t] = s0[t]; ((double2 *)(ws.qea + FD_PAD))[t] = s3[t]; ((double2 *)(ws.qeg + FD_PAD))[t] = s4[t];
                }
                for (int t = lane; t < mq; t += 32) ws.u.a.qk[t] = key_hi(P.seed, (unsigned long long)(hq.pix0 + t));
                // (the keys share their storage with the drain tables, so p's keys are rebuilt for every pair)
                for (int t = lane; t < mp; t += 32) ws.u.a.pk[t] = key_lo(P.seed, (unsigned long long)(hp.pix0 + t));
                if (lane < FD_PAD) {
                    const int j = FD_PAD + 2 * npad2 + lane;
                    ws.qc[j] = LYA_CHI_SENTINEL; ws.qea[j] = 0.0; ws.qeg[j] = 0.0;
                }
            }
            __syncwarp();
            // per row of p: in-grid window [jlo, jhi) of q and the sign change jx (chi_i >= chi_j below it)
            const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;
            const double Tchi = (s > 0.0) ? (bp.rperp_max / s) * (1.0 + 1e-12) + 1e-9 : 1e300;
            for (int i = lane; i < mp; i += 32) {
                const double x = ws.pc[i];
                int lo = 0, hi = mq;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (qc[mid] > x - R) hi = mid; else lo = mid + 1; }
                const int jlo = lo;
                const double top = fmin(x + R, Tchi - x);
                hi = mq;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (qc[mid] >= top) hi = mid; else lo = mid + 1; }
                const int jhi = lo;
                lo = jlo; hi = jhi;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (qc[mid] > x) hi = mid; else lo = mid + 1; }
                ws.jlo[i] = (unsigned char)jlo; ws.jhi[i] = (unsigned char)jhi; ws.jx[i] = (unsigned char)lo;
            }
            __syncwarp();
            // ---- pass A ----
            unsigned binned = 0, kept_n = 0;
            for (int i0 = 0; i0 < mp; i0 += FD_ROWS) {
                const int i = i0 + lane;
                int plo = 1 << 20, phi = -(1 << 20), nlo = 1 << 20, nhi = -(1 << 20), r0 = 1 << 20, r1 = -1;
                if (lane < FD_ROWS && i < mp) {
                    const int jl = ws.jlo[i], jh = ws.jhi[i], jx = ws.jx[i];
                    if (jx > jl) { plo = jl - i; phi = jx - 1 - i; }
                    if (jh > jx) { nlo = jx - i; nhi = jh - 1 - i; }
                    if (jh > jl) { r0 = i; r1 = i; }
                }
                plo = __reduce_min_sync(0xffffffffu, plo); phi = __reduce_max_sync(0xffffffffu, phi);
                nlo = __reduce_min_sync(0xffffffffu, nlo); nhi = __reduce_max_sync(0xffffffffu, nhi);
                r0 = __reduce_min_sync(0xffffffffu, r0); r1 = __reduce_max_sync(0xffffffffu, r1);
                if (r1 < r0) continue;
#pragma unroll 1
                for (int sgn = 0; sgn >= -1; --sgn)         // one call site: chi_i >= chi_j, then chi_i < chi_j
                    dm_walk_any<POW2>(ws, h01, h23, r0 & ~1, r1 | 1, mq, sgn ? nlo : plo, sgn ? nhi : phi, sgn, bp, g,
                                      (unsigned)c0, np1, P.thr, lane, binned, kept_n, evaluated);
            }
            binned_total += binned; kept_total += kept_n;
            __syncwarp();
            // ---- pass B: compact the non-zero entries (H_aa > 0 wherever a pair with weight fell) ----
            int nnz = 0;
            for (int t0 = 0; t0 < n_slots; t0 += 32) {
                const int t = t0 + lane;
                bool nzf = false;
                if (t < n_slots) {
                    const int cr = t / (int)np1, bx = t - cr * (int)np1;
                    const double2 a = ws.H01[t], b = ws.H23[t];
                    nzf = (bx < bp.n_par) && (cr < LYA_NCOL) && (a.x != 0.0 || a.y != 0.0 || b.x != 0.0 || b.y != 0.0);
                }
                const unsigned bal = __ballot_sync(0xffffffffu, nzf);
                if (nzf) ws.u.b.nz[nnz + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)t;
                nnz += __popc(bal);
            }
            __syncwarp();
            // ---- pass C (one drain call site: the kernel's code has to stay small for the instruction cache) ----
            // Normally the queue holds every kept pair.  With more kept pairs than the queue holds (small
            // reject fractions) the mask is redone row by row and the queue drained each time it fills.
            const unsigned nk = ws.nkept;
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
                        int A = -1;
                        if (j < jh) A = lya_pix_bin_t<POW2>(bp, g, ws.pc[si], qc[j]);
                        const bool kp = (A >= 0) && keep_pair(key_lo(P.seed, (unsigned long long)(hp.pix0 + si)),
                                                              key_hi(P.seed, (unsigned long long)(hq.pix0 + j)), P.thr);   // (the staged keys are gone)
                        const unsigned bal = __ballot_sync(0xffffffffu, kp);
                        if (n_q + __popc(bal) > FD_KCAP) break;          // drain first, then redo these 32 pixels
                        if (kp) ws.kept[n_q + __popc(bal & ((1u << lane) - 1u))] = ((unsigned)si << 20) | ((unsigned)j << 12) | (unsigned)A;
                        n_q += __popc(bal);
                        sj += 32;
                    }
                    done = si >= mp;
                }
                __syncwarp();
                dm_drain<POW2>(ws, n_q, nnz, mp, mq, P, g, c0, hp.off, hq.off, lane, n_red);
                __syncwarp();
                if (done) break;
                n_q = 0;
            }
            __syncwarp();
            // clear the table and the queue for the next pair
            for (int t = lane; t < n_slots; t += 32) { ws.H01[t] = make_double2(0.0, 0.0); ws.H23[t] = make_double2(0.0, 0.0); }
            if (lane == 0) ws.nkept = 0u;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
        kept_total += __shfl_xor_sync(0xffffffffu, kept_total, o);
        binned_total += __shfl_xor_sync(0xffffffffu, binned_total, o);
        n_red += __shfl_xor_sync(0xffffffffu, n_red, o);
    }
    if (lane == 0) {
        atomicAdd(&P.counters[2], evaluated);
        atomicAdd(&P.counters[5], kept_total);
        atomicAdd(&P.counters[6], binned_total);
        atomicAdd(&P.counters[7], n_red);
    }
}

// Dn_t, Wd_t: accumulators in transposed bin order.  Writes the API-order outputs (any may be NULL):
// D[A][B] = Dn[A][B] / Wd[A] (row 0 where Wd[A] == 0), Dn, Wd.
__global__ void k_dmat_normalise(const double *Dn_t, const double *Wd_t, BinParams bp, double *D, double *Dn, double *Wd)
{
    const int nb = bp.n_par * bp.n_perp;
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= (int64_t)nb * nb) return;
    const int A = (int)(idx / nb), B = (int)(idx - (int64_t)A * nb);
    const int ax = A / bp.n_perp, ay = A - ax * bp.n_perp, bx = B / bp.n_perp, by = B - bx * bp.n_perp;
    const int At = ay * bp.n_par + ax, Bt = by * bp.n_par + bx;
    const double wd = Wd_t[At], v = Dn_t[(size_t)At * nb + Bt];
    if (D) D[idx] = (wd != 0.0) ? v / wd : 0.0;
    if (Dn) Dn[idx] = v;
    if (Wd && B == 0) Wd[A] = wd;
}

// API-order version for already-summed numerators: D[A][B] = Dn[A][B] / Wd[A] (row 0 where Wd[A] == 0)
__global__ void k_dmat_divide(const double *Dn, const double *Wd, int nb, double *D)
{
    const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= (int64_t)nb * nb) return;
    const double wd = Wd[idx / nb];
    D[idx] = (wd != 0.0) ? Dn[idx] / wd : 0.0;
}

}  // namespace

namespace {
__global__ void k_fp_flag(const int32_t *pq, int64_t n, unsigned long long seed, unsigned long long thr, unsigned *flag)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int2 e = ((const int2 *)pq)[k];
    const unsigned long long lo = (unsigned long long)min(e.x, e.y), hi = (unsigned long long)max(e.x, e.y);
    flag[k] = keep_pair(key_lo(seed, lo), key_hi(seed, hi), thr) ? 1u : 0u;
}
__global__ void k_fp_compact(const int32_t *pq, int64_t n, const unsigned *flag, const unsigned long long *pos, int32_t *out)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n || !flag[k]) return;
    ((int2 *)out)[pos[k]] = ((const int2 *)pq)[k];
}
}  // namespace

extern "C" lya_status lya_pairs_subsample(lya_ctx *ctx, const lya_pairs *pairs, double reject_fraction, uint64_t seed,
                                          lya_pairs **out, int64_t *n_kept)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pairs || !out || !n_kept) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_pairs_subsample: NULL argument");
    if (!(reject_fraction >= 0.0 && reject_fraction <= 1.0))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_pairs_subsample: reject_fraction must be in [0,1]");
    *out = NULL; *n_kept = 0;
    LYA_CUDA(cudaSetDevice(ctx->device));
    lya_pairs *pl = (lya_pairs *)calloc(1, sizeof(lya_pairs));
    if (!pl) return lya_fail(ctx, LYA_ERR_OOM, "host allocation failed");
    const int64_t n = pairs->n;
    if (n == 0) { *out = pl; return LYA_OK; }
    double t = floor(reject_fraction * 4294967296.0 + 0.5);
    if (t < 0) t = 0;
    if (t > 4294967296.0) t = 4294967296.0;
    const unsigned long long thr = (unsigned long long)t;
    cudaStream_t s = ctx->stream;
    unsigned *flag = NULL;
    unsigned long long *pos = NULL, *tmp = NULL;
    cudaError_t e = cudaMalloc(&flag, sizeof(unsigned) * (size_t)n);
    if (e == cudaSuccess) e = cudaMalloc(&pos, sizeof(unsigned long long) * (size_t)(n + 1));
    if (e == cudaSuccess) e = cudaMalloc(&tmp, sizeof(unsigned long long) * (size_t)(n / 2048 + 4));
    auto drop = [&]() { cudaFree(flag); cudaFree(pos); cudaFree(tmp); };
    if (e != cudaSuccess) { drop(); free(pl); return lya_cuda_fail(ctx, e, "cudaMalloc(lya_pairs_subsample)"); }
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_fp_flag<<<blocks, 256, 0, s>>>(pairs->pq, n, seed, thr, flag);
    e = lya_exclusive_scan(flag, pos, n, tmp, s);
    unsigned long long total = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&total, pos + n, sizeof(total), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { drop(); free(pl); return lya_cuda_fail(ctx, e, "lya_pairs_subsample"); }
    pl->n = (int64_t)total;
    if (total > 0) {
        e = cudaMalloc(&pl->pq, sizeof(int32_t) * 2 * (size_t)total);
        if (e == cudaSuccess) {
            k_fp_compact<<<blocks, 256, 0, s>>>(pairs->pq, n, flag, pos, pl->pq);
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        }
        if (e != cudaSuccess) { if (pl->pq) cudaFree(pl->pq); drop(); free(pl); return lya_cuda_fail(ctx, e, "lya_pairs_subsample"); }
    }
    drop();
    *out = pl; *n_kept = pl->n;
    return LYA_OK;
}

extern "C" lya_status lya_dmat(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                               double reject_fraction, uint64_t seed, double *D, double *Dn_out, double *Wd_out,
                               lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pairs) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: pairs is NULL");
    if (!D && !Dn_out) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: need D or Dn");
    if (!(reject_fraction >= 0.0 && reject_fraction <= 1.0))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: reject_fraction must be in [0,1]");
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    if (b->n_par > H_SLOTS) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: n_par above %d", H_SLOTS);
    if ((int64_t)b->n_par * b->n_perp > 4096) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: more than 4096 bins");
    st = lya_check_forests_host(ctx, f, true, false, true);
    if (st) return st;
    if (f->n_forest > 0 && !(f->ux && f->uy && f->uz))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat needs ux,uy,uz (device)");
    LYA_CUDA(cudaSetDevice(ctx->device));
    int max_len = 0;
    st = lya_validate_forests(ctx, f, false, true, &max_len);
    if (st) return st;

    const int nb = b->n_par * b->n_perp;
    cudaStream_t s = ctx->stream;
    const BinParams bp = lya_make_binparams(b);
    const bool use_fast = pairs->n > 0 && (b->n_par + 1) * LYA_NCOL <= FD_SLOTS && b->n_perp + 2 <= 256 &&
                          !ctx->force_generic;
    double *scal = NULL, *Dn = NULL, *Wd = NULL;          // internal accumulators (transposed bin order)
    bool own_Dn = false, own_Wd = false;
    const int64_t nf = f->n_forest;
    LyaPrep prep;
    LyaBuckets bk;
    memset(&prep, 0, sizeof(prep));
    memset(&bk, 0, sizeof(bk));
    auto cleanup = [&]() { cudaFree(scal); if (own_Dn) cudaFree(Dn); if (own_Wd) cudaFree(Wd); lya_prep_free(&prep); lya_buckets_free(&bk); };
    cudaEventRecord(ctx->ev[3], s);
    if (use_fast) {
        st = lya_prep_build(ctx, f, false, true, &prep);
        if (st) return st;
        cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
        st = lya_bucket_pairs(ctx, &prep, &bp, pairs, 0, &bk);
        if (st) { cleanup(); return st; }
        if (bk.bad_pair == LYA_DEV_DEGENERATE) { cleanup(); return lya_fail(ctx, LYA_ERR_DEGENERATE_FOREST, "a listed forest has sum w == 0 or sum w (L-Lbar)^2 == 0"); }
        if (bk.bad_pair) { cleanup(); return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)"); }
    }
    cudaError_t e = cudaMalloc(&scal, sizeof(double) * 3 * (size_t)(nf ? nf : 1));
    if (e == cudaSuccess && !Dn) { e = cudaMalloc(&Dn, sizeof(double) * (size_t)nb * nb); own_Dn = (e == cudaSuccess); if (!own_Dn) Dn = NULL; }
    if (e == cudaSuccess && !Wd) { e = cudaMalloc(&Wd, sizeof(double) * (size_t)nb); own_Wd = (e == cudaSuccess); if (!own_Wd) Wd = NULL; }
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "cudaMalloc(lya_dmat)"); }
    cudaMemsetAsync(Dn, 0, sizeof(double) * (size_t)nb * nb, s);
    cudaMemsetAsync(Wd, 0, sizeof(double) * (size_t)nb, s);
    cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
    unsigned long long thr;
    {
        double t = floor(reject_fraction * 4294967296.0 + 0.5);
        if (t < 0) t = 0;
        if (t > 4294967296.0) t = 4294967296.0;
        thr = (unsigned long long)t;
    }
    // generic kernel (long forests, wide column span, fine pixel spacing): original arrays
    DmParams P;
    P.pix_off = f->pix_off; P.chi = f->chi; P.w = f->w; P.loglam = f->loglam;
    P.ux = f->ux; P.uy = f->uy; P.uz = f->uz;
    P.f_invS = scal; P.f_lbar = scal + nf; P.f_invV = scal + 2 * nf;
    P.pq = use_fast ? bk.pq + 2 * bk.n_fast : pairs->pq;
    P.n_pairs = use_fast ? bk.n_generic : pairs->n;
    P.n_forest = nf;
    P.bp = bp;
    P.seed = seed; P.thr = thr;
    P.Dn = Dn; P.Wd = Wd; P.counters = ctx->d_counters;
    P.LC = H_SLOTS / b->n_par;
    if (P.LC > 8) P.LC = 8;
    if (P.LC > b->n_perp) P.LC = b->n_perp;

    cudaEventRecord(ctx->ev[0], s);
    if (use_fast && bk.n_fast > 0) {
        DmFastParams F;
        F.prep = prep; F.pq = bk.pq; F.n_pairs = bk.n_fast; F.bp = bp; F.seed = seed; F.thr = thr;
        F.Dn = Dn; F.Wd = Wd; F.counters = ctx->d_counters;
        const size_t fsmem = sizeof(DmFastWarp) * FD_WARPS;
        const int fgrid = ctx->sm_count;
        if (bp.pow2) {
            e = cudaFuncSetAttribute(k_dmat_fast<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem);
            if (e == cudaSuccess) k_dmat_fast<true><<<fgrid, FD_THREADS, fsmem, s>>>(F);
        } else {
            e = cudaFuncSetAttribute(k_dmat_fast<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem);
            if (e == cudaSuccess) k_dmat_fast<false><<<fgrid, FD_THREADS, fsmem, s>>>(F);
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_dmat_fast launch"); }
    }
    if (P.n_pairs > 0) {
        k_forest_scalars<<<(unsigned)((nf + 127) / 128), 128, 0, s>>>(f->pix_off, f->w, f->loglam, nf, scal, scal + nf, scal + 2 * nf);
        const size_t smem = sizeof(DmWarpSmem) * DM_WARPS;
        int grid = ctx->sm_count * 2;
        if (P.bp.pow2) {
            e = cudaFuncSetAttribute(k_dmat<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) k_dmat<true><<<grid, DM_THREADS, smem, s>>>(P);
        } else {
            e = cudaFuncSetAttribute(k_dmat<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) k_dmat<false><<<grid, DM_THREADS, smem, s>>>(P);
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_dmat launch"); }
    }
    cudaEventRecord(ctx->ev[1], s);
    k_dmat_normalise<<<(unsigned)(((int64_t)nb * nb + 255) / 256), 256, 0, s>>>(Dn, Wd, bp, D, Dn_out, Wd_out);
    cudaEventRecord(ctx->ev[2], s);
    unsigned long long h[8];
    e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_dmat"); }
    const unsigned long long visited = use_fast ? bk.visited : h[1];
    cleanup();
    switch ((unsigned)h[3]) {
    case LYA_DEV_OK: break;
    case LYA_DEV_DEGENERATE: return lya_fail(ctx, LYA_ERR_DEGENERATE_FOREST, "a listed forest has sum w == 0 or sum w (L-Lbar)^2 == 0");
    case LYA_DEV_TOO_LONG: return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: a listed forest has more than %d pixels", DTILE);
    default: return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
    }
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_forest_pairs = (uint64_t)pairs->n;
        stats->n_visited = visited;
        stats->n_evaluated = h[2];
        stats->n_kept = h[5];
        stats->n_binned = h[6];
        stats->n_scatter = h[7];
        cudaEventElapsedTime(&stats->ms_main, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&stats->ms_total, ctx->ev[3], ctx->ev[2]);
    }
    return LYA_OK;
}

extern "C" lya_status lya_dmat_normalise(lya_ctx *ctx, const lya_binning *b, const double *Dn, const double *Wd, double *D)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    if (!Dn || !Wd || !D) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat_normalise: NULL argument");
    LYA_CUDA(cudaSetDevice(ctx->device));
    const int nb = b->n_par * b->n_perp;
    k_dmat_divide<<<(unsigned)(((int64_t)nb * nb + 255) / 256), 256, 0, ctx->stream>>>(Dn, Wd, nb, D);
    LYA_CUDA(cudaGetLastError());
    return LYA_OK;
}
