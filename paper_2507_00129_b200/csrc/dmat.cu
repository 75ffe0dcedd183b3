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
#include "lya_walk.cuh"

namespace {

constexpr int DM_WARPS = 4;
constexpr int DM_THREADS = DM_WARPS * 32;
constexpr int DTILE = 128;               // max pixels per forest handled by this kernel
constexpr int DQPAD = 4;
constexpr int H_SLOTS = 512;             // local (b_par, column) slots per H table
constexpr int KEPT_CAP = 256;
constexpr int DCHUNK = 8;

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
    double sw = 0.0, swl = 0.0;                               // Lbar = L_0 + sum w (L - L_0) / sum w (exact differences: prep.cu)
    const double l0 = (b > a) ? loglam[a] : 0.0;
    for (int64_t k = a; k < b; ++k) { sw += w[k]; swl += w[k] * (loglam[k] - l0); }
    double lb = (sw > 0.0) ? l0 + swl / sw : 0.0;
    double v = 0.0;
    for (int64_t k = a; k < b; ++k) { double u = loglam[k] - lb; v += w[k] * u * u; }
    const double tiny = 1e-12 * fabs(lb);                  // reading R-7: all weighted L equal up to rounding of L - Lbar
    bool ok = (sw > 0.0) && (v > sw * tiny * tiny);
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
                    ws.pk[t] = lya_key_lo(P.seed, (unsigned long long)(op + ip0 + t));
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
                    if (in) ws.qk[j] = lya_key_hi(P.seed, (unsigned long long)(oq + jq0 + j));
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
                                bool kp = (bin >= 0) && lya_keep_pair(ki, ws.qk[min(j, mq - 1)], P.thr);
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

#include "dmat_fast.cuh"
#include "dmat_long.cuh"

namespace {
__global__ void k_fp_flag(const int32_t *pq, int64_t n, unsigned long long seed, unsigned long long thr, unsigned *flag)
{
    const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int2 e = ((const int2 *)pq)[k];
    const unsigned long long lo = (unsigned long long)min(e.x, e.y), hi = (unsigned long long)max(e.x, e.y);
    flag[k] = lya_keep_pair(lya_key_lo(seed, lo), lya_key_hi(seed, hi), thr) ? 1u : 0u;
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
    LYA_CUDA(lya_enter(ctx));
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
    cudaError_t e = lya_malloc(&flag, sizeof(unsigned) * (size_t)n);
    if (e == cudaSuccess) e = lya_malloc(&pos, sizeof(unsigned long long) * (size_t)(n + 1));
    if (e == cudaSuccess) e = lya_malloc(&tmp, sizeof(unsigned long long) * (size_t)(n / 2048 + 4));
    auto drop = [&]() { lya_free(flag); lya_free(pos); lya_free(tmp); };
    if (e != cudaSuccess) { drop(); free(pl); return lya_cuda_fail(ctx, e, "lya_malloc(lya_pairs_subsample)"); }
    const unsigned blocks = (unsigned)((n + 255) / 256);
    { k_fp_flag<<<blocks, 256, 0, s>>>(pairs->pq, n, seed, thr, flag); lya_note_launch(); }
    e = lya_exclusive_scan(flag, pos, n, tmp, s);
    unsigned long long total = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&total, pos + n, sizeof(total), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { drop(); free(pl); return lya_cuda_fail(ctx, e, "lya_pairs_subsample"); }
    pl->n = (int64_t)total;
    if (total > 0) {
        e = lya_malloc(&pl->pq, sizeof(int32_t) * 2 * (size_t)total);
        if (e == cudaSuccess) {
            { k_fp_compact<<<blocks, 256, 0, s>>>(pairs->pq, n, flag, pos, pl->pq); lya_note_launch(); }
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        }
        if (e != cudaSuccess) { if (pl->pq) lya_free(pl->pq); drop(); free(pl); return lya_cuda_fail(ctx, e, "lya_pairs_subsample"); }
    }
    drop();
    *out = pl; *n_kept = pl->n;
    return LYA_OK;
}

static lya_status dmat_run(lya_ctx *ctx, const lya_plan *pl, double reject_fraction, uint64_t seed,
                           double *D, double *Dn_out, double *Wd_out, lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pl) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: plan is NULL");
    if (!pl->has_dmat) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: the plan was created without want_dmat");
    if (!D && !Dn_out) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: need D or Dn");
    if (!(reject_fraction >= 0.0 && reject_fraction <= 1.0))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: reject_fraction must be in [0,1]");
    const lya_forests *f = &pl->f;
    const lya_binning *b = &pl->b;
    if (b->n_par > H_SLOTS) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: n_par above %d", H_SLOTS);
    if (pl->listed_degenerate)
        return lya_fail(ctx, LYA_ERR_DEGENERATE_FOREST, "a listed forest has sum w == 0 or sum w (L-Lbar)^2 == 0");
    LYA_CUDA(lya_enter(ctx));

    const int nb = b->n_par * b->n_perp;
    cudaStream_t s = ctx->stream;
    const BinParams bp = pl->bp;
    const bool use_fast = pl->use_fast;
    const LyaBuckets &bk = pl->bk;
    double *scal = NULL, *Dn = NULL, *Wd = NULL;          // internal accumulators (transposed bin order)
    const int64_t nf = f->n_forest;
    auto cleanup = [&]() { lya_free(scal); lya_free(Dn); lya_free(Wd); };
    cudaEventRecord(ctx->ev[3], s);
    cudaError_t e = lya_malloc(&scal, sizeof(double) * 3 * (size_t)(nf ? nf : 1));
    if (e == cudaSuccess) e = lya_malloc(&Dn, sizeof(double) * (size_t)nb * nb);
    if (e == cudaSuccess) e = lya_malloc(&Wd, sizeof(double) * (size_t)nb);
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_malloc(lya_dmat)"); }
    cudaMemsetAsync(Dn, 0, sizeof(double) * (size_t)nb * nb, s);
    cudaMemsetAsync(Wd, 0, sizeof(double) * (size_t)nb, s);
    cudaMemsetAsync(ctx->d_counters, 0, 16 * sizeof(unsigned long long), s);
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
    P.pq = use_fast ? bk.pq + 2 * (bk.n_fast + bk.n_fast2 + bk.n_long) : pl->pq;
    P.n_pairs = use_fast ? bk.n_generic : pl->n_pairs;
    P.n_forest = nf;
    P.bp = bp;
    P.seed = seed; P.thr = thr;
    P.Dn = Dn; P.Wd = Wd; P.counters = ctx->d_counters;
    P.LC = H_SLOTS / b->n_par;
    if (P.LC > 8) P.LC = 8;
    if (P.LC > b->n_perp) P.LC = b->n_perp;

    cudaEventRecord(ctx->ev[0], s);
    if (use_fast && bk.n_fast + bk.n_fast2 + bk.n_long > 0) {
        DmFastParams F;
        F.prep = pl->prep; F.bp = bp; F.seed = seed; F.thr = thr;
        F.Dn = Dn; F.Wd = Wd; F.counters = ctx->d_counters;
        const int fgrid = ctx->sm_count;
        auto launch = [&](auto kern, int threads, size_t fsmem) {
            cudaError_t le = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem);
            if (le == cudaSuccess) { kern<<<fgrid, threads, fsmem, s>>>(F); lya_note_launch(); }
            return le;
        };
        e = cudaSuccess;
        if (bk.n_fast > 0) {                                  // class 0: forests of up to 72 pixels, spacing above the bin width
            F.pq = bk.pq; F.n_pairs = bk.n_fast;
            const int th = DmCfg<0>::WARPS * 32;
            const size_t sm = DmPool<0>::SMEM_BYTES;
            if (ctx->check_holders) e = bp.pow2 ? launch(k_dmat_fast<true, true, 0>, th, sm) : launch(k_dmat_fast<false, true, 0>, th, sm);
            else e = bp.pow2 ? launch(k_dmat_fast<true, false, 0>, th, sm) : launch(k_dmat_fast<false, false, 0>, th, sm);
        }
        if (e == cudaSuccess && bk.n_fast2 > 0) {             // class 1: up to 144 pixels, diagonal stride up to 8
            // (its own work counter: counters[4] is reset between the two launches on the stream)
            cudaMemsetAsync(ctx->d_counters + 4, 0, sizeof(unsigned long long), s);
            F.pq = bk.pq + 2 * bk.n_fast; F.n_pairs = bk.n_fast2;
            const int th = DmCfg<1>::WARPS * 32;
            const size_t sm = DmPool<1>::SMEM_BYTES;
            if (ctx->check_holders) e = bp.pow2 ? launch(k_dmat_fast<true, true, 1>, th, sm) : launch(k_dmat_fast<false, true, 1>, th, sm);
            else e = bp.pow2 ? launch(k_dmat_fast<true, false, 1>, th, sm) : launch(k_dmat_fast<false, false, 1>, th, sm);
        }
        if (e == cudaSuccess && bk.n_long > 0) {              // long forests: up to 1024 pixels, one CTA per forest pair
            cudaMemsetAsync(ctx->d_counters + 4, 0, sizeof(unsigned long long), s);
            F.pq = bk.pq + 2 * (bk.n_fast + bk.n_fast2); F.n_pairs = bk.n_long;
            if (ctx->check_holders) e = bp.pow2 ? launch(k_dmat_long<true, true>, DL_THREADS, DL_SMEM_BYTES) : launch(k_dmat_long<false, true>, DL_THREADS, DL_SMEM_BYTES);
            else e = bp.pow2 ? launch(k_dmat_long<true, false>, DL_THREADS, DL_SMEM_BYTES) : launch(k_dmat_long<false, false>, DL_THREADS, DL_SMEM_BYTES);
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_dmat_fast launch"); }
    }
    if (P.n_pairs > 0) {
        { k_forest_scalars<<<(unsigned)((nf + 127) / 128), 128, 0, s>>>(f->pix_off, f->w, f->loglam, nf, scal, scal + nf, scal + 2 * nf); lya_note_launch(); }
        const size_t smem = sizeof(DmWarpSmem) * DM_WARPS;
        int grid = ctx->sm_count * 2;
        if (P.bp.pow2) {
            e = cudaFuncSetAttribute(k_dmat<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) { k_dmat<true><<<grid, DM_THREADS, smem, s>>>(P); lya_note_launch(); }
        } else {
            e = cudaFuncSetAttribute(k_dmat<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) { k_dmat<false><<<grid, DM_THREADS, smem, s>>>(P); lya_note_launch(); }
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_dmat launch"); }
    }
    cudaEventRecord(ctx->ev[1], s);
    { k_dmat_normalise<<<(unsigned)(((int64_t)nb * nb + 255) / 256), 256, 0, s>>>(Dn, Wd, bp, D, Dn_out, Wd_out); lya_note_launch(); }
    cudaEventRecord(ctx->ev[2], s);
    unsigned long long h[16];
    e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_dmat"); }
    const unsigned long long visited = use_fast ? pl->visited : h[1];
    cleanup();
    switch ((unsigned)h[3]) {
    case LYA_DEV_OK: break;
    case LYA_DEV_DEGENERATE: return lya_fail(ctx, LYA_ERR_DEGENERATE_FOREST, "a listed forest has sum w == 0 or sum w (L-Lbar)^2 == 0");
    case LYA_DEV_TOO_LONG: return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: a listed forest has more than %d pixels", DTILE);
    default: return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
    }
    if (h[10] != 0)
        return lya_fail(ctx, LYA_ERR_CUDA, "k_dmat_fast: %llu table entries had two holders (LYA_OPT_CHECK_HOLDERS)", h[10]);
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_forest_pairs = (uint64_t)pl->n_pairs;
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

extern "C" lya_status lya_dmat_plan(lya_ctx *ctx, const lya_plan *plan, double reject_fraction, uint64_t seed,
                                    double *D, double *Dn, double *Wd, lya_stats *stats)
{
    return dmat_run(ctx, plan, reject_fraction, seed, D, Dn, Wd, stats);
}

extern "C" lya_status lya_dmat(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                               double reject_fraction, uint64_t seed, double *D, double *Dn_out, double *Wd_out,
                               lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!D && !Dn_out) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: need D or Dn");
    if (!(reject_fraction >= 0.0 && reject_fraction <= 1.0))
        return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat: reject_fraction must be in [0,1]");
    if (b && (int64_t)b->n_par * b->n_perp > 4096) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: more than 4096 bins");
    lya_plan *pl = NULL;
    lya_status st = lya_plan_create(ctx, f, b, pairs, 0, 1, &pl);
    if (st) return st;
    st = dmat_run(ctx, pl, reject_fraction, seed, D, Dn_out, Wd_out, stats);
    lya_plan_free(ctx, pl);
    return st;
}

extern "C" lya_status lya_dmat_normalise(lya_ctx *ctx, const lya_binning *b, const double *Dn, const double *Wd, double *D)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    if (!Dn || !Wd || !D) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_dmat_normalise: NULL argument");
    LYA_CUDA(lya_enter(ctx));
    const int nb = b->n_par * b->n_perp;
    { k_dmat_divide<<<(unsigned)(((int64_t)nb * nb + 255) / 256), 256, 0, ctx->stream>>>(Dn, Wd, nb, D); lya_note_launch(); }
    LYA_CUDA(cudaGetLastError());
    return LYA_OK;
}
