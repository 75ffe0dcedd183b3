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
// One warp per forest pair.  Pass 1a: diagonal walk with register run-length
// accumulation of (H_aa, H_ag, H_ga, H_gg) into a warp-private shared-memory table
// indexed by (b_par, b_perp - c0).  Pass 1b: every in-grid pair is hashed (stage 4
// mask, pure integer); kept pairs are queued in shared memory and drained by the whole
// warp: T1-T4 go to the L2-resident Dn with red.global.add.f64.
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
    unsigned long long *counters;   // [0] next chunk, [1] visited, [2] evaluated, [3] error, [4] kept, [5] binned
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
};

__device__ __forceinline__ void red_add(double *addr, double v) { atomicAdd(addr, v); }

// Drain the kept-pair queue: T1..T3 (first column chunk only) and T4 (this chunk's columns).
template <bool POW2>
__device__ void drain_kept(DmWarpSmem &ws, int n_kept, int mp, int mq, const DmParams &P, const PairBin &g,
                           double invSp, double invVp, double invSq, double invVq,
                           int c0, int ncol, bool first_chunk, int lane)
{
    const BinParams &bp = P.bp;
    const int nb = bp.n_par * bp.n_perp;
    const double *qc = ws.qc + DQPAD, *qw = ws.qw + DQPAD, *qu = ws.qu + DQPAD;
    for (int e = 0; e < n_kept; ++e) {
        const unsigned rec = ws.kept[e];
        const int i = rec >> 20, j = (rec >> 12) & 0xff, A = rec & 0xfff;
        const double om = ws.pw[i] * qw[j];
        const double ui = ws.pu[i], uj = qu[j];
        double *row = P.Dn + (size_t)A * nb;
        if (first_chunk) {
            if (lane == 0) { red_add(row + A, om); red_add(P.Wd + A, om); }
            for (int j2 = lane; j2 < mq; j2 += 32) {                       // T2
                int B = lya_pix_bin<POW2>(bp, g, ws.pc[i], qc[j2]);
                if (B >= 0) {
                    double aj = qw[j2] * invSq, gj = qw[j2] * qu[j2] * invVq;
                    red_add(row + B, -om * (aj + uj * gj));
                }
            }
            for (int i2 = lane; i2 < mp; i2 += 32) {                       // T3
                int B = lya_pix_bin<POW2>(bp, g, ws.pc[i2], qc[j]);
                if (B >= 0) {
                    double ai = ws.pw[i2] * invSp, gi = ws.pw[i2] * ws.pu[i2] * invVp;
                    red_add(row + B, -om * (ai + ui * gi));
                }
            }
        }
        const int n_slots = bp.n_par * ncol;                               // T4
        for (int t = lane; t < n_slots; t += 32) {
            double haa = ws.H[0][t];
            if (haa != 0.0 || ws.H[3][t] != 0.0 || ws.H[1][t] != 0.0 || ws.H[2][t] != 0.0) {
                int bx = t / ncol, lc = t - bx * ncol;
                int B = bx * bp.n_perp + c0 + lc;
                double v = haa + uj * ws.H[1][t] + ui * ws.H[2][t] + ui * uj * ws.H[3][t];
                red_add(row + B, om * v);
            }
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
    int cur_p = -1;
    double invSp = 0, invVp = 0;
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
            const int mp = (int)(P.pix_off[p + 1] - op), mq = (int)(P.pix_off[q + 1] - oq);
            if (mp == 0 || mq == 0) continue;
            if (mp > DTILE || mq > DTILE) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_TOO_LONG);
                continue;
            }
            const double invSq = P.f_invS[q], invVq = P.f_invV[q], lbq = P.f_lbar[q];
            __syncwarp();
            if (p != cur_p) {
                invSp = P.f_invS[p]; invVp = P.f_invV[p];
                const double lbp = P.f_lbar[p];
                for (int t = lane; t < mp; t += 32) {
                    ws.pc[t] = P.chi[op + t];
                    ws.pw[t] = P.w[op + t];
                    ws.pu[t] = P.loglam[op + t] - lbp;
                    ws.pk[t] = key_lo(P.seed, (unsigned long long)(op + t));
                }
                cur_p = p;
            }
            if (isnan(invSp) || isnan(invVp) || isnan(invSq) || isnan(invVq)) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_DEGENERATE);
                continue;
            }
            for (int t = lane; t < mq + 2 * DQPAD; t += 32) {
                int j = t - DQPAD;
                bool in = (j >= 0) && (j < mq);
                ws.qc[t] = in ? P.chi[oq + j] : LYA_CHI_SENTINEL;
                ws.qw[t] = in ? P.w[oq + j] : 0.0;
                ws.qu[t] = in ? P.loglam[oq + j] - lbq : 0.0;
                if (in) ws.qk[j] = key_hi(P.seed, (unsigned long long)(oq + j));
            }
            __syncwarp();
            visited += (unsigned long long)mp * mq;
            double s, c;
            lya_pair_sc(P.ux[p], P.uy[p], P.uz[p], P.ux[q], P.uy[q], P.uz[q], s, c);
            const PairBin g = lya_make_pairbin(bp, s, c);

            // r_perp column range of this forest pair: r_perp is increasing in both pixels
            int c_first, c_last;
            {
                double t0 = __dmul_rn(__dadd_rn(ws.pc[0], qc[0]), g.s);
                double t1 = __dmul_rn(__dadd_rn(ws.pc[mp - 1], qc[mq - 1]), g.s);
                if (!(t0 < bp.rperp_max)) continue;                        // nothing in the grid
                c_first = min((int)lya_floor_u32(__dmul_rn(t0, bp.inv_perp)), bp.n_perp - 1);
                c_last = (t1 < bp.rperp_max) ? min((int)lya_floor_u32(__dmul_rn(t1, bp.inv_perp)), bp.n_perp - 1)
                                             : bp.n_perp - 1;
            }
            for (int c0 = c_first; c0 <= c_last; c0 += LC) {
                const int ncol = min(LC, c_last - c0 + 1);
                const bool first_chunk = (c0 == c_first);
                const int n_slots = bp.n_par * ncol;
                for (int t = lane; t < n_slots; t += 32) { ws.H[0][t] = 0.0; ws.H[1][t] = 0.0; ws.H[2][t] = 0.0; ws.H[3][t] = 0.0; }
                __syncwarp();
                // ---- pass 1a: H tables; lanes own diagonals d = j - i, register run-length ----
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
                __syncwarp();
                // ---- pass 1b: mask every in-grid pair, queue the kept ones, drain ----
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
                                drain_kept<POW2>(ws, n_q, mp, mq, P, g, invSp, invVp, invSq, invVq, c0, ncol, first_chunk, lane);
                                __syncwarp();
                                n_q = 0;
                            }
                            if (kp) ws.kept[n_q + __popc(bal & ((1u << lane) - 1u))] = ((unsigned)i << 20) | ((unsigned)j << 12) | (unsigned)bin;
                            n_q += __popc(bal);
                        }
                    }
                }
                __syncwarp();
                drain_kept<POW2>(ws, n_q, mp, mq, P, g, invSp, invVp, invSq, invVq, c0, ncol, first_chunk, lane);
                __syncwarp();
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
        atomicAdd(&P.counters[4], kept_total);
        atomicAdd(&P.counters[5], binned);
    }
}

__global__ void k_dmat_normalise(const double *Dn, const double *Wd, int nb, double *D)
{
    int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= (int64_t)nb * nb) return;
    double wd = Wd[idx / nb];
    D[idx] = (wd != 0.0) ? Dn[idx] / wd : 0.0;
}

}  // namespace

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
    if (max_len > 255) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_dmat: forests longer than 255 pixels are not supported yet");

    const int nb = b->n_par * b->n_perp;
    cudaStream_t s = ctx->stream;
    double *scal = NULL, *Dn = Dn_out, *Wd = Wd_out;
    bool own_Dn = false, own_Wd = false;
    const int64_t nf = f->n_forest;
    LYA_CUDA(cudaMalloc(&scal, sizeof(double) * 3 * (size_t)(nf ? nf : 1)));
    if (!Dn) { cudaError_t e = cudaMalloc(&Dn, sizeof(double) * (size_t)nb * nb); if (e != cudaSuccess) { cudaFree(scal); return lya_cuda_fail(ctx, e, "cudaMalloc(Dn)"); } own_Dn = true; }
    if (!Wd) { cudaError_t e = cudaMalloc(&Wd, sizeof(double) * (size_t)nb); if (e != cudaSuccess) { cudaFree(scal); if (own_Dn) cudaFree(Dn); return lya_cuda_fail(ctx, e, "cudaMalloc(Wd)"); } own_Wd = true; }
    auto cleanup = [&]() { cudaFree(scal); if (own_Dn) cudaFree(Dn); if (own_Wd) cudaFree(Wd); };
    cudaMemsetAsync(Dn, 0, sizeof(double) * (size_t)nb * nb, s);
    cudaMemsetAsync(Wd, 0, sizeof(double) * (size_t)nb, s);
    cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
    if (nf > 0)
        k_forest_scalars<<<(unsigned)((nf + 127) / 128), 128, 0, s>>>(f->pix_off, f->w, f->loglam, nf, scal, scal + nf, scal + 2 * nf);

    DmParams P;
    P.pix_off = f->pix_off; P.chi = f->chi; P.w = f->w; P.loglam = f->loglam;
    P.ux = f->ux; P.uy = f->uy; P.uz = f->uz;
    P.f_invS = scal; P.f_lbar = scal + nf; P.f_invV = scal + 2 * nf;
    P.pq = pairs->pq; P.n_pairs = pairs->n; P.n_forest = nf;
    P.bp = lya_make_binparams(b);
    P.seed = seed;
    {
        double t = floor(reject_fraction * 4294967296.0 + 0.5);
        if (t < 0) t = 0;
        if (t > 4294967296.0) t = 4294967296.0;
        P.thr = (unsigned long long)t;
    }
    P.Dn = Dn; P.Wd = Wd; P.counters = ctx->d_counters;
    P.LC = H_SLOTS / b->n_par;
    if (P.LC > 8) P.LC = 8;
    if (P.LC > b->n_perp) P.LC = b->n_perp;

    const size_t smem = sizeof(DmWarpSmem) * DM_WARPS;
    cudaEventRecord(ctx->ev[0], s);
    if (pairs->n > 0) {
        cudaError_t e;
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
    if (D) k_dmat_normalise<<<(unsigned)(((int64_t)nb * nb + 255) / 256), 256, 0, s>>>(Dn, Wd, nb, D);
    cudaEventRecord(ctx->ev[2], s);
    unsigned long long h[8];
    cudaError_t e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_dmat"); }
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
        stats->n_visited = h[1];
        stats->n_evaluated = h[2];
        stats->n_kept = h[4];
        stats->n_binned = h[5];
        cudaEventElapsedTime(&stats->ms_main, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&stats->ms_total, ctx->ev[0], ctx->ev[2]);
    }
    return LYA_OK;
}
