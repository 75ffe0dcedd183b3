// xi2pcf.cu -- stage 2 (lya_xi2pcf): the pair kernel of eq. 2.4.
//
//   S_A = sum (w_i d_i)(w_j d_j),  W_A = sum w_i w_j,  N_A = #pairs,  xi_A = S_A / W_A
// over pixel pairs (i in p, j in q) of the listed forest pairs whose separation
// r_par = |chi_i - chi_j| c, r_perp = (chi_i + chi_j) s falls in bin A.
//
// Design (B200): persistent grid, one WARP per forest pair.
//   * the forest-pair list is bucket-sorted by the r_perp column of the pair's first
//     pixels (prep.cu); all bins of a pair lie in columns [c0, c0 + LYA_NCOL), so every
//     warp keeps a PRIVATE (n_par x LYA_NCOL) sub-histogram in shared memory that lives
//     across thousands of forest pairs and is merged into the global fp64/u64
//     accumulators (red.global) only when the warp moves to another bucket;
//   * both forests are staged in shared memory from the padded catalogue with 16-byte
//     loads (forest p is reused across the consecutive pairs that share it);
//   * lanes own DIAGONALS d = j - i of the (i, j) pixel-pair matrix (1, 2 or 4 adjacent ones per
//     lane, sliding register window over q).  Along a diagonal r_par is nearly constant and
//     r_perp grows slowly, so consecutive pairs fall in the same bin: a lane works on a RUN and
//     touches the sub-histogram only when the bin changes;
//   * B200 has no native shared-memory fp64 (or 64-bit) atomic add -- they compile to a CAS loop.
//     The fast kernel needs none: the lanes of one row step hold pixel pairs (i, j_lane) with the
//     same i and distinct j, which fall in distinct bins on each side of chi_i = chi_j when q's
//     pixel spacing exceeds the r_par bin width (the two sides have their own rows), so every
//     entry has one lane working on it and that lane simply HOLDS the entry (S, W, N) in registers,
//     storing it back and loading the next one with predicated st/ld.shared when its bin changes.
//     Pairs that break the assumption (and long forests, wide column spans) go to the generic
//     kernel below, which uses CAS atomics on a block-level histogram;
//   * only rows/diagonals that can hold an in-grid pair are walked: two binary searches per row of p
//     on the increasing chi of q give the window (r_par band and r_perp cut), and the matrix is
//     walked 16 rows at a time over exactly the diagonals those rows need.
// Geometry is exact binary64, operation by operation (lya_internal.cuh), so N is
// bit-identical to the oracle for any traversal order.
#include <stdlib.h>
#include "lya_walk.cuh"

namespace {

// ======================= generic kernel: any forest length, any column span =======================
// Block-level histogram with CAS atomics; pairs come from the ORIGINAL arrays.
constexpr int XI_WARPS = 8;                 // warps per block
constexpr int XI_THREADS = XI_WARPS * 32;
constexpr int TILE = 128;                   // pixels of a forest staged per tile
constexpr int QPAD = 8;                     // sentinel slots either side of the q tile
constexpr int CHUNK = 16;                   // forest pairs claimed per atomic
constexpr unsigned long long WARP_BUDGET = 1ull << 28;   // visited pairs per warp per launch (u32 N safety)

struct XiParams {
    const int64_t *pix_off;
    const double *chi, *w, *delta;
    const double *ux, *uy, *uz;
    const int32_t *pq;
    int64_t n_pairs;
    int64_t n_forest;
    BinParams bp;
    double *S, *W;                    // global accumulators [nb]
    unsigned long long *N;            // [nb]
    unsigned long long *counters;     // [0] next chunk, [1] visited, [2] evaluated, [3] error flag
};

struct WarpSmem {
    double pc[TILE], pa[TILE], pw[TILE];
    double qc[TILE + 2 * QPAD], qa[TILE + 2 * QPAD], qw[TILE + 2 * QPAD];
};

__device__ __forceinline__ void flush_run(double *sS, double *sW, unsigned *sN, int bin, double accS, double accW, unsigned cnt)
{
    atomicAdd(&sN[bin], cnt);
    atomicAdd(&sS[bin], accS);
    atomicAdd(&sW[bin], accW);
}

// One tile (mp x mq pixels, already staged) of one forest pair, D diagonals per lane.
template <int D, bool POW2>
__device__ __forceinline__ void tile_diagonals(const WarpSmem &ws, int mp, int mq, int dlo, int dhi,
                                               const BinParams &bp, const PairBin &g,
                                               double *sS, double *sW, unsigned *sN, int lane,
                                               unsigned long long &evaluated)
{
    const double *qc = ws.qc + QPAD, *qa = ws.qa + QPAD, *qw = ws.qw + QPAD;
    for (int d0 = dlo; d0 <= dhi; d0 += 32 * D) {
        const int dl = d0 + lane * D;                       // first diagonal of this lane
        const int dpass_hi = min(dhi, d0 + 32 * D - 1);
        int i_begin = max(0, -dpass_hi);
        int i_end = min(mp, mq - d0);                       // exclusive
        if (i_end <= i_begin) continue;
        // round the trip count up to a multiple of D (extra rows hit p padding = sentinel-free
        // but masked by row validity below)
        int cur[D]; double accS[D], accW[D]; unsigned cnt[D];
        double wc[D], wa[D], ww[D];                         // sliding window over q
#pragma unroll
        for (int k = 0; k < D; ++k) { cur[k] = -1; accS[k] = 0.0; accW[k] = 0.0; cnt[k] = 0; }
        // preload window slots 0..D-2 with q[i_begin + dl + k]
#pragma unroll
        for (int k = 0; k < D - 1; ++k) {
            int j = min(max(i_begin + dl + k, -QPAD), mq + QPAD - 1);
            wc[k] = qc[j]; wa[k] = qa[j]; ww[k] = qw[j];
        }
        evaluated += (unsigned long long)(i_end - i_begin) * D;
        for (int ib = i_begin; ib < i_end; ib += D) {
#pragma unroll
            for (int u = 0; u < D; ++u) {
                const int i = ib + u;
                if (i < i_end) {                            // warp-uniform
                    const double pci = ws.pc[i], pai = ws.pa[i], pwi = ws.pw[i];
                    {   // new q pixel for the last diagonal of the lane goes into slot (u + D - 1) % D
                        int j = min(max(i + dl + D - 1, -QPAD), mq + QPAD - 1);
                        wc[(u + D - 1) % D] = qc[j]; wa[(u + D - 1) % D] = qa[j]; ww[(u + D - 1) % D] = qw[j];
                    }
#pragma unroll
                    for (int k = 0; k < D; ++k) {
                        const int sl = (k + u) % D;         // slot holding q[i + dl + k]
                        const int bin = lya_pix_bin<POW2>(bp, g, pci, wc[sl]);
                        if (bin != cur[k]) {
                            if (cur[k] >= 0) flush_run(sS, sW, sN, cur[k], accS[k], accW[k], cnt[k]);
                            cur[k] = bin; accS[k] = 0.0; accW[k] = 0.0; cnt[k] = 0;
                        }
                        if (bin >= 0) {
                            accS[k] = fma(pai, wa[sl], accS[k]);
                            accW[k] = fma(pwi, ww[sl], accW[k]);
                            cnt[k] += 1;
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int k = 0; k < D; ++k)
            if (cur[k] >= 0) flush_run(sS, sW, sN, cur[k], accS[k], accW[k], cnt[k]);
    }
}

template <int D, bool POW2>
__global__ void __launch_bounds__(XI_THREADS, 2) k_xi(XiParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nb = P.bp.n_par * P.bp.n_perp;
    double *sS = (double *)smem_raw;
    double *sW = sS + nb;
    unsigned *sN = (unsigned *)(sW + nb);
    WarpSmem *wsm = (WarpSmem *)(smem_raw + (((size_t)nb * 20 + 15) & ~(size_t)15));
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    WarpSmem &ws = wsm[wid];

    for (int k = threadIdx.x; k < nb; k += XI_THREADS) { sS[k] = 0.0; sW[k] = 0.0; sN[k] = 0u; }
    __syncthreads();

    const BinParams bp = P.bp;
    unsigned long long visited = 0, evaluated = 0;
    int cur_p = -1, cur_ip0 = -1;
    const int64_t n_chunks = (P.n_pairs + CHUNK - 1) / CHUNK;
    // conservative half-width of the r_par window in chi: |chi_i - chi_j| * c < rpar_max
    while (visited < WARP_BUDGET) {
        unsigned long long chunk = 0;
        if (lane == 0) chunk = atomicAdd(&P.counters[0], 1ull);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if ((int64_t)chunk >= n_chunks) break;
        const int64_t k0 = (int64_t)chunk * CHUNK, k1 = min(k0 + CHUNK, P.n_pairs);
        for (int64_t k = k0; k < k1; ++k) {
            const int p = P.pq[2 * k], q = P.pq[2 * k + 1];
            if ((unsigned)p >= (unsigned)P.n_forest || (unsigned)q >= (unsigned)P.n_forest) {
                if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_BAD_PAIR);
                continue;
            }
            const int64_t op = P.pix_off[p], oq = P.pix_off[q];
            const int np = (int)(P.pix_off[p + 1] - op), nq = (int)(P.pix_off[q + 1] - oq);
            if (np == 0 || nq == 0) continue;
            visited += (unsigned long long)np * nq;
            double s, c;
            lya_pair_sc(P.ux[p], P.uy[p], P.uz[p], P.ux[q], P.uy[q], P.uz[q], s, c);
            const PairBin g = lya_make_pairbin(bp, s, c);
            // chi window: r_par < rpar_max  <=>  |dchi| < rpar_max / c  (margin: conservative superset)
            const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;

            for (int ip0 = 0; ip0 < np; ip0 += TILE) {
                const int mp = min(TILE, np - ip0);
                if (p != cur_p || ip0 != cur_ip0) {
                    __syncwarp();
                    for (int t = lane; t < mp; t += 32) {
                        double wv = P.w[op + ip0 + t];
                        ws.pc[t] = P.chi[op + ip0 + t];
                        ws.pw[t] = wv;
                        ws.pa[t] = wv * P.delta[op + ip0 + t];
                    }
                    cur_p = p; cur_ip0 = ip0;
                }
                for (int jq0 = 0; jq0 < nq; jq0 += TILE) {
                    const int mq = min(TILE, nq - jq0);
                    __syncwarp();
                    for (int t = lane; t < mq + 2 * QPAD; t += 32) {
                        int j = t - QPAD;
                        bool in = (j >= 0) && (j < mq);
                        double wv = in ? P.w[oq + jq0 + j] : 0.0;
                        ws.qc[t] = in ? P.chi[oq + jq0 + j] : LYA_CHI_SENTINEL;
                        ws.qw[t] = wv;
                        ws.qa[t] = in ? wv * P.delta[oq + jq0 + j] : 0.0;
                    }
                    __syncwarp();
                    // diagonal range [dlo, dhi] of rows with a non-empty r_par window (exact, from
                    // per-row binary searches; chi_q is increasing)
                    int dlo = 1 << 30, dhi = -(1 << 30);
                    const double *qc = ws.qc + QPAD;
                    for (int i = lane; i < mp; i += 32) {
                        const double x = ws.pc[i];
                        int lo = 0, hi = mq;                 // first j with qc[j] > x - R
                        while (lo < hi) { int mid = (lo + hi) >> 1; if (qc[mid] > x - R) hi = mid; else lo = mid + 1; }
                        int jlo = lo;
                        lo = jlo; hi = mq;                   // first j with qc[j] >= x + R
                        while (lo < hi) { int mid = (lo + hi) >> 1; if (qc[mid] >= x + R) hi = mid; else lo = mid + 1; }
                        int jhi = lo;
                        if (jhi > jlo) { dlo = min(dlo, jlo - i); dhi = max(dhi, jhi - 1 - i); }
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        dlo = min(dlo, __shfl_xor_sync(0xffffffffu, dlo, o));
                        dhi = max(dhi, __shfl_xor_sync(0xffffffffu, dhi, o));
                    }
                    if (dhi >= dlo)
                        tile_diagonals<D, POW2>(ws, mp, mq, dlo, dhi, bp, g, sS, sW, sN, lane, evaluated);
                }
            }
        }
    }
    // warp counters
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
    if (lane == 0) {
        atomicAdd(&P.counters[1], visited);
        atomicAdd(&P.counters[2], evaluated);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nb; k += XI_THREADS) {
        unsigned n = sN[k];
        if (n) {
            atomicAdd(&P.N[k], (unsigned long long)n);
            atomicAdd(&P.S[k], sS[k]);
            atomicAdd(&P.W[k], sW[k]);
        }
    }
}

// Sub-sample mode (NEXT-1), pairs the fast kernel cannot take: one warp per forest pair, lanes over
// the pixel pairs, global atomics into the accumulators of the pair's sub-sample.  Slow and simple.
template <bool POW2>
__global__ void k_xi_direct(XiParams P, const int32_t *region)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const BinParams bp = P.bp;
    const int nb = bp.n_par * bp.n_perp;
    unsigned long long visited = 0;
    for (int64_t k = warp; k < P.n_pairs; k += n_warps) {
        const int p = P.pq[2 * k], q = P.pq[2 * k + 1];
        if ((unsigned)p >= (unsigned)P.n_forest || (unsigned)q >= (unsigned)P.n_forest) {
            if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_BAD_PAIR);
            continue;
        }
        const int64_t op = P.pix_off[p], oq = P.pix_off[q];
        const int64_t np = P.pix_off[p + 1] - op, nq = P.pix_off[q + 1] - oq;
        if (np == 0 || nq == 0) continue;
        visited += (unsigned long long)(np * nq);
        double s, c;
        lya_pair_sc(P.ux[p], P.uy[p], P.uz[p], P.ux[q], P.uy[q], P.uz[q], s, c);
        const PairBin g = lya_make_pairbin(bp, s, c);
        const size_t roff = (size_t)(region ? region[p] : 0) * nb;
        for (int64_t t = lane; t < np * nq; t += 32) {
            const int64_t i = t / nq, j = t - i * nq;
            const int A = lya_pix_bin<POW2>(bp, g, P.chi[op + i], P.chi[oq + j]);
            if (A >= 0) {
                const double wi = P.w[op + i], wj = P.w[oq + j];
                atomicAdd(&P.S[roff + A], (wi * P.delta[op + i]) * (wj * P.delta[oq + j]));
                atomicAdd(&P.W[roff + A], wi * wj);
                atomicAdd(&P.N[roff + A], 1ull);
            }
        }
    }
    if (lane == 0 && visited) { atomicAdd(&P.counters[1], visited); atomicAdd(&P.counters[2], visited); }
}

__global__ void k_xi_finalize(const double *S, const double *W, const unsigned long long *N, int nb,
                              double *S_out, double *W_out, unsigned long long *N_out, double *xi_out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nb) return;
    double s = S[k], w = W[k];
    if (S_out) S_out[k] = s;
    if (W_out) W_out[k] = w;
    if (N_out) N_out[k] = N[k];
    if (xi_out) xi_out[k] = (w != 0.0) ? s / w : 0.0;
}

template <int D>
cudaError_t launch_xi(const XiParams &P, int grid, size_t smem, cudaStream_t s)
{
    cudaError_t e;
    if (P.bp.pow2) {
        e = cudaFuncSetAttribute(k_xi<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        { k_xi<D, true><<<grid, XI_THREADS, smem, s>>>(P); lya_note_launch(); }
    } else {
        e = cudaFuncSetAttribute(k_xi<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        { k_xi<D, false><<<grid, XI_THREADS, smem, s>>>(P); lya_note_launch(); }
    }
    return cudaGetLastError();
}

// ======================= fast kernel: warp-private sub-histograms ================================
// Two size classes (template parameter CLS), as in k_dmat_fast:
//   class 0: forests of up to LYA_FAST_TILE (72) pixels whose spacing exceeds the r_par bin width -- the BASELINE
//            configs; 14 warps per SM (16.2 KB of shared memory per warp);
//   class 1: forests of up to LYA_FAST_TILE2 (144) pixels, spacing down to bin width / 8 -- native-resolution shapes
//            (NEXT-3): one diagonal per lane at a DIAGONAL STRIDE ds (the lanes of a row step sit ds pixels of q
//            apart, so they still hold different r_par bins on each side); 11 warps per SM (19.6 KB per warp).
template <int CLS> struct XiCfg;
template <> struct XiCfg<0> { static constexpr int T = LYA_FAST_TILE, WARPS = 14; };
template <> struct XiCfg<1> { static constexpr int T = LYA_FAST_TILE2, WARPS = 11; };
constexpr int FW = XiCfg<0>::WARPS;          // (class 0 under its old names: the no-allocation entry point uses them)
constexpr int FTHREADS = FW * 32;
constexpr int FT = LYA_FAST_TILE;            // longest forest (pixels)
#ifndef LYA_FROWS
#define LYA_FROWS 24
#endif
constexpr int FROWS = LYA_FROWS;             // rows of p walked per pass (keeps lanes busy: DESIGN.md)
static_assert(FROWS % 12 == 0 && FROWS <= 32, "a row group holds whole blocks of 1, 2, 3 or 4 rows");
constexpr int FTP = ((FT + 15) / 16) * 16 + 2;   // p rows incl. sentinel rows
constexpr int FPAD = 2;                      // sentinel pixels either side of q (reads are clamped)
constexpr int FSLOTS = 612;                  // 2 * (n_par + 1) * LYA_NCOL <= FSLOTS
constexpr int FCHUNK = 16;                   // forest pairs claimed per atomic

struct XiFastParams {
    LyaPrep prep;
    const int32_t *pq;
    int64_t n_pairs;
    BinParams bp;
    double *S, *W;
    unsigned long long *N;
    unsigned long long *counters;            // [4] next chunk, [2] evaluated
    const int32_t *region;                   // NULL, or the sub-sample (sky region) of every forest (NEXT-1)
    int n_region;
    unsigned long long merge_every;          // visited pixel pairs after which a warp merges its sub-histogram (u32 counters)
};

// Sub-histogram slot = col_rel * 2 (n_par + 1) + side * (n_par + 1) + row.
//   side: 0 when chi_i >= chi_j, 1 otherwise (the two sides of a bin are added when the warp merges);
//   row n_par is GARBAGE: a pixel pair outside the grid (or a sentinel pixel) maps to entry
//   (column 0, side 0, row n_par), so the pair loop has no validity branch; the merge drops that row.
template <int T_> struct __align__(16) FastWarpT {
    static constexpr int T = T_, TP = ((T_ + 15) / 16) * 16 + 2;   // longest forest; p rows incl. sentinel rows
    double2 SW[FSLOTS];                      // (S, W) per slot
    unsigned N[(FSLOTS + 3) & ~3];           // (padded: the arrays below need 16-byte alignment)
    double pc[TP], pa[TP], pw[TP];           // rows >= len are sentinels (walks cover whole row groups)
    double qc[T_ + 2 * FPAD], qa[T_ + 2 * FPAD], qw[T_ + 2 * FPAD];
    unsigned char jlo[T_], jhi[T_];          // per row of p: window [jlo, jhi) of q that can be in the grid
};
using FastWarp = FastWarpT<FT>;
static_assert(sizeof(FastWarpT<LYA_FAST_TILE>) * XiCfg<0>::WARPS <= 232448 && sizeof(FastWarpT<LYA_FAST_TILE2>) * XiCfg<1>::WARPS <= 232448, "k_xi_fast shared memory");

// (predicated shared-memory accesses: lya_walk.cuh)

// byte offset (16 * slot) of a pixel pair's sub-histogram entry
template <bool POW2>
__device__ __forceinline__ unsigned xi_key(const BinParams &bp, const PairBin &g, double chi_i, double chi_j, unsigned c0,
                                           unsigned np1)
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
    const unsigned side = (unsigned)__double2hiint(d) >> 31;
    const unsigned off = ((col * 2u + side) * np1 + bx) << 4;
    unsigned key;                                                           // outside the window -> the garbage entry (0, 0, n_par)
    asm("{\n .reg .pred v;\n setp.lt.u32 v, %1, %2;\n setp.lt.and.u32 v, %3, %4, v;\n selp.u32 %0, %5, %6, v;\n}"
        : "=r"(key) : "r"(bx), "r"(np1 - 1u), "r"(col), "r"((unsigned)LYA_NCOL), "r"(off), "r"((np1 - 1u) << 4));
    return key;
}

// Walk rows [r0, r1] of p against the diagonals [dlo, dhi], D adjacent diagonals per lane.
// Each lane HOLDS the sub-histogram entry (S, W, N) of its current run in registers: when the key
// changes it stores the entry back (release) and loads the new one (acquire), both predicated, so the
// loop has no divergent branch.  The lanes of a row hold pixel pairs (i, j_lane) with distinct j on
// their side of chi_i = chi_j, hence distinct entries (lya_pair_key: q's spacing exceeds the r_par bin
// width), so an entry has one holder at a time; all releases of a row come before its acquires (warp
// barrier in between).  The keys of row i+1 are computed between the acquire of row i and the FMAs
// that need it.  r1 - r0 + 1 is a multiple of D; rows >= mp of p are sentinels.
// AL2 (D == 2 only, first row even, dlo even): the new q pixels of the two rows of a loop step are neighbours at an
// even index, so ONE 16-byte read per array serves both rows -- and unlike the 8-byte reads at a stride of two
// pixels it has no bank conflict.
// ds (D == 1 only; 1 otherwise): diagonal stride -- blocks of 32 * ds diagonals, ds passes per block (one per
// residue), lane l on diagonal d0 + ds * l.
template <int D, bool POW2, bool CHECK, bool AL2 = false, class WS>
__device__ __forceinline__ void xi_walk(WS &ws, unsigned sw_base, unsigned n_base, int r0, int r1, int mq,
                                        int dlo, int dhi, const BinParams &bp, const PairBin &g, unsigned c0,
                                        unsigned np1, int lane, unsigned long long &evaluated, unsigned &conflicts, int ds = 1)
{
    const double *qc = ws.qc + FPAD, *qa = ws.qa + FPAD, *qw = ws.qw + FPAD;
    const unsigned garbage = (np1 - 1u) * 16u;              // entry (column 0, side 0, row n_par)
    const int step = (D == 1) ? ds : D, n_res = (D == 1) ? ds : 1;
    const int n_pass = ((dhi - dlo) / (32 * step) + 1) * n_res;
    for (int pass = 0; pass < n_pass; ++pass) {
        const int d0 = dlo + (pass / n_res) * (32 * step) + pass % n_res;
        if (d0 > dhi) continue;
        const int dl = d0 + lane * step;                    // first diagonal of this lane
        unsigned cur[D], cnt[D], key[D];
        double accS[D], accW[D], fa[D], fw[D];
        double wc[D], wa[D], ww[D];                         // sliding window over q
        double pa_c, pw_c;
        double2 qc2 = make_double2(0.0, 0.0), qa2 = qc2, qw2 = qc2;   // AL2: the q pixels of rows ib + 1 and ib + 2
#pragma unroll
        for (int k = 0; k < D; ++k) { cur[k] = garbage; cnt[k] = 0u; accS[k] = 0.0; accW[k] = 0.0; }
        {   // prologue: window and keys of row r0
#pragma unroll
            for (int k = 0; k < D; ++k) {
                const int j = min(max(r0 + dl + k, -FPAD), mq + FPAD - 1);
                wc[k] = qc[j]; wa[k] = qa[j]; ww[k] = qw[j];
            }
            const double pci = ws.pc[r0];
            pa_c = ws.pa[r0]; pw_c = ws.pw[r0];
#pragma unroll
            for (int k = 0; k < D; ++k) { key[k] = xi_key<POW2>(bp, g, pci, wc[k], c0, np1); fa[k] = wa[k]; fw[k] = ww[k]; }
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
                                if (other == key[k] && key[k] != garbage && key[k] != garbage + np1 * 16u &&   // (row n_par of either side is garbage)
                                    (src < lane || (src == lane && k2 < k))) conflicts += 1u;
                        }
                }
                // row i + 1's new q pixel and p pixel are read BEFORE the hand-over (they do not depend on it; the
                // volatile accesses below would otherwise pin these loads behind them)
                double qcn, qan, qwn;
                if (AL2) {
                    if (u == 0) {                           // (even index: 16-byte aligned; beyond either end -> two sentinels)
                        const unsigned jc = min((unsigned)(i + dl + D + FPAD), (unsigned)((mq + 3) & ~1));
                        qc2 = *(const double2 *)&ws.qc[jc]; qa2 = *(const double2 *)&ws.qa[jc]; qw2 = *(const double2 *)&ws.qw[jc];
                    }
                    qcn = u == 0 ? qc2.x : qc2.y; qan = u == 0 ? qa2.x : qa2.y; qwn = u == 0 ? qw2.x : qw2.y;
                } else {
                    const unsigned jn = min((unsigned)(i + dl + D + FPAD), (unsigned)(mq + 2 * FPAD - 1));
                    qcn = ws.qc[jn]; qan = ws.qa[jn]; qwn = ws.qw[jn];
                }
                const double pcn = ws.pc[i + 1];
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    ch[k] = key[k] != cur[k];
                    sts_v2_if(ch[k], sw_base + cur[k], accS[k], accW[k]);                 // release
                    sts_u32_if(ch[k], n_base + (cur[k] >> 2), cnt[k]);
                }
                __syncwarp();
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    lds_v2_if(ch[k], sw_base + key[k], accS[k], accW[k]);                 // acquire
                    lds_u32_if(ch[k], n_base + (key[k] >> 2), cnt[k]);
                    cur[k] = key[k];
                }
                // row i + 1: its new q pixel replaces q[i + dl] in window slot u
                double fa_n[D], fw_n[D];
                unsigned key_n[D];
                {
                    // (one unsigned min clamps both ends: a negative index wraps to the right-hand sentinel)
                    wc[u] = qcn; wa[u] = qan; ww[u] = qwn;
                    const double pci = pcn;
#pragma unroll
                    for (int k = 0; k < D; ++k) {
                        const int sl = (k + u + 1) % D;
                        key_n[k] = xi_key<POW2>(bp, g, pci, wc[sl], c0, np1);
                        fa_n[k] = wa[sl]; fw_n[k] = ww[sl];
                    }
                }
#pragma unroll
                for (int k = 0; k < D; ++k) {
                    accS[k] = fma(pa_c, fa[k], accS[k]);
                    accW[k] = fma(pw_c, fw[k], accW[k]);
                    cnt[k] += 1u;
                    fa[k] = fa_n[k]; fw[k] = fw_n[k]; key[k] = key_n[k];
                }
                pa_c = ws.pa[i + 1]; pw_c = ws.pw[i + 1];
            }
        }
        // release what the lanes still hold
#pragma unroll
        for (int k = 0; k < D; ++k) {
            sts_v2_if(true, sw_base + cur[k], accS[k], accW[k]);
            sts_u32_if(true, n_base + (cur[k] >> 2), cnt[k]);
        }
        __syncwarp();
    }
}

template <bool POW2, bool CHECK, class WS>
__device__ __forceinline__ void xi_walk_any(WS &ws, unsigned sw_base, unsigned n_base, int i0, int r0, int r1, int mq,
                                            int dlo, int dhi, const BinParams &bp, const PairBin &g, unsigned c0,
                                            unsigned np1, int lane, unsigned long long &evaluated, unsigned &conflicts, int ds)
{
    // D diagonals per lane, the smallest that covers the group in one pass; the rows [r0, r1] (inside one group of
    // FROWS rows, i0 its first) are widened to a multiple of D rows aligned to the group
    const int nd = dhi - dlo + 1;
    if (ds > 1) {                                            // pixels finer than the bins: one diagonal per lane, ds apart
        xi_walk<1, POW2, CHECK>(ws, sw_base, n_base, r0, r1, mq, dlo, dhi, bp, g, c0, np1, lane, evaluated, conflicts, ds);
        return;
    }
#define XI_WALK_D(D_) do { const int a = i0 + ((r0 - i0) / D_) * D_, b = a + ((r1 - a) / D_ + 1) * D_ - 1; \
        xi_walk<D_, POW2, CHECK>(ws, sw_base, n_base, a, b, mq, dlo, dhi, bp, g, c0, np1, lane, evaluated, conflicts); } while (0)
    if (nd <= 32) XI_WALK_D(1);
    else if (nd <= 64 && dhi - (dlo - (dlo & 1)) <= 63) {    // two diagonals per lane from an EVEN first diagonal (AL2);
        const int a = i0 + ((r0 - i0) / 2) * 2, b = a + ((r1 - a) / 2 + 1) * 2 - 1;          // 64 diagonals from an odd one take D = 3
        xi_walk<2, POW2, CHECK, true>(ws, sw_base, n_base, a, b, mq, dlo - (dlo & 1), dhi, bp, g, c0, np1, lane, evaluated, conflicts);
    }
    else if (nd <= 96) XI_WALK_D(3);
    else XI_WALK_D(4);
#undef XI_WALK_D
}

// merge a warp's sub-histogram (first column c0) into the global accumulators and clear it
template <class WS>
__device__ __forceinline__ void xi_merge(WS &ws, const XiFastParams &P, int c0, int reg, int lane)
{
    const size_t roff = (size_t)reg * (size_t)(P.bp.n_par * P.bp.n_perp);   // accumulators of sub-sample reg
    const int np1 = P.bp.n_par + 1;
    __syncwarp();
    for (int t = lane; t < np1 * LYA_NCOL; t += 32) {            // t = col_rel * np1 + row
        const int cr = t / np1, bx = t - cr * np1, col = c0 + cr;
        const int s0 = cr * 2 * np1 + bx, s1 = s0 + np1;          // the two sides of the bin
        const unsigned n = ws.N[s0] + ws.N[s1];
        if (n) {
            if (bx < P.bp.n_par && cr < LYA_NCOL && col < P.bp.n_perp) {
                const double2 v0 = ws.SW[s0], v1 = ws.SW[s1];
                const int A = bx * P.bp.n_perp + col;
                atomicAdd(&P.N[roff + A], (unsigned long long)n);
                atomicAdd(&P.S[roff + A], v0.x + v1.x);
                atomicAdd(&P.W[roff + A], v0.y + v1.y);
            }
            ws.N[s0] = 0u; ws.N[s1] = 0u;
        }
        ws.SW[s0] = make_double2(0.0, 0.0); ws.SW[s1] = make_double2(0.0, 0.0);
    }
    __syncwarp();
}

template <bool POW2, bool CHECK, int CLS = 0>
__global__ void __launch_bounds__(XiCfg<CLS>::WARPS * 32, 1) k_xi_fast(XiFastParams P)
{
    using WS = FastWarpT<XiCfg<CLS>::T>;
    constexpr int FTP = WS::TP;                                // (shadows the class-0 constant)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    WS &ws = ((WS *)smem_raw)[wid];
    const BinParams bp = P.bp;
    const unsigned np1 = (unsigned)bp.n_par + 1u;
    for (int t = lane; t < FSLOTS; t += 32) { ws.SW[t] = make_double2(0.0, 0.0); ws.N[t] = 0u; }
    if (lane < FPAD) { ws.qc[lane] = LYA_CHI_SENTINEL; ws.qa[lane] = 0.0; ws.qw[lane] = 0.0; }
    __syncwarp();

    const double *qc = ws.qc + FPAD;
    const unsigned sw_base = (unsigned)__cvta_generic_to_shared(ws.SW), n_base = (unsigned)__cvta_generic_to_shared(ws.N);
    unsigned long long evaluated = 0, since_merge = 0;
    unsigned conflicts = 0;
    int cur_p = -1, head_p = -1, win_c0 = -1, win_reg = 0;
    ForestHead hp;
    hp.len = 0;
    const int64_t n_chunks = (P.n_pairs + FCHUNK - 1) / FCHUNK;
    for (;;) {
        unsigned long long chunk = 0;
        if (lane == 0) chunk = atomicAdd(&P.counters[4], 1ull);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if ((int64_t)chunk >= n_chunks) break;
        const int64_t k0 = (int64_t)chunk * FCHUNK, k1 = min(k0 + FCHUNK, P.n_pairs);
        // the chunk's list entries in one coalesced read (lane l holds entry k0 + l), and the 80-byte records of its
        // q forests on their way into L1 while the first pairs are worked on (the chain list entry -> record ->
        // pixel arrays was three dependent L2 round trips per forest pair)
        int2 e_l = make_int2(0, 0);
        if (lane < (int)(k1 - k0)) {
            e_l = ((const int2 *)P.pq)[k0 + lane];
            const char *hq_addr = (const char *)(P.prep.head + e_l.y);
            asm volatile("prefetch.global.L1 [%0];" :: "l"(hq_addr));
            asm volatile("prefetch.global.L1 [%0];" :: "l"(hq_addr + sizeof(ForestHead) - 1));
        }
        for (int64_t k = k0; k < k1; ++k) {
            const int2 e = make_int2(__shfl_sync(0xffffffffu, e_l.x, (int)(k - k0)), __shfl_sync(0xffffffffu, e_l.y, (int)(k - k0)));
            const int p = e.x, q = e.y;
            if (p != head_p) { hp = P.prep.head[p]; head_p = p; }
            const ForestHead hq = P.prep.head[q];
            const int mp = hp.len, mq = hq.len;
            double s, c;
            lya_pair_sc(hp.ux, hp.uy, hp.uz, hq.ux, hq.uy, hq.uz, s, c);
            const PairBin g = lya_make_pairbin(bp, s, c);
            int c0;
            const int key = lya_pair_key<POW2>(bp, g, hp, hq, c0);
            if (key >= (CLS + 1) * bp.n_perp || key < CLS * bp.n_perp) continue;     // cannot happen in this class's range
            const int ds = (CLS == 0) ? 1 : lya_pair_stride(bp, g, hq);                // lanes of a row step sit ds pixels of q apart
            since_merge += (unsigned long long)mp * mq;
            const int reg = P.region ? P.region[p] : 0;       // a pixel pair belongs to the sub-sample of forest p
            if (c0 != win_c0 || reg != win_reg || since_merge > P.merge_every) {
                if (win_c0 >= 0) xi_merge(ws, P, win_c0, win_reg, lane);
                win_c0 = c0; win_reg = reg; since_merge = (unsigned long long)mp * mq;
            }
            __syncwarp();
            if (p != cur_p) {
                const double2 *sc = (const double2 *)(P.prep.chi + hp.off), *sa = (const double2 *)(P.prep.a + hp.off),
                              *sw = (const double2 *)(P.prep.w + hp.off);
                for (int t = lane; 2 * t < mp; t += 32) {
                    ((double2 *)ws.pc)[t] = sc[t]; ((double2 *)ws.pa)[t] = sa[t]; ((double2 *)ws.pw)[t] = sw[t];
                }
                __syncwarp();
                for (int t = mp + lane; t < FTP; t += 32) {              // sentinel rows (!= q's sentinel: r_par never 0)
                    ws.pc[t] = 2.0 * LYA_CHI_SENTINEL; ws.pa[t] = 0.0; ws.pw[t] = 0.0;
                }
                cur_p = p;
            }
            {
                const double2 *sc = (const double2 *)(P.prep.chi + hq.off), *sa = (const double2 *)(P.prep.a + hq.off),
                              *sw = (const double2 *)(P.prep.w + hq.off);
                const int npad2 = (mq + 1) >> 1;
                for (int t = lane; t < npad2; t += 32) {
                    ((double2 *)qc)[t] = sc[t]; ((double2 *)(ws.qa + FPAD))[t] = sa[t]; ((double2 *)(ws.qw + FPAD))[t] = sw[t];
                }
                if (lane < FPAD) {                           // right sentinels (the pad pixel of an odd forest is one already)
                    const int j = 2 * npad2 + lane;
                    ws.qc[FPAD + j] = LYA_CHI_SENTINEL; ws.qa[FPAD + j] = 0.0; ws.qw[FPAD + j] = 0.0;
                }
            }
            __syncwarp();
            // per row of p: the window of q with r_par < rpar_max and r_perp < rperp_max (conservative superset)
            const double R = (c > 0.0) ? (bp.rpar_max / c) * (1.0 + 1e-12) + 1e-9 : 1e300;
            const double Tchi = (s > 0.0) ? (bp.rperp_max / s) * (1.0 + 1e-12) + 1e-9 : 1e300;
            // (branch-free lower bounds of fixed trip count, two rows per lane: four independent chains in flight
            //  instead of two data-dependent loops one after the other; qc[mq] is a sentinel, so a probe past the
            //  end reads "true" and the position never exceeds mq)
            for (int ib = 0; ib < mp; ib += 64) {
                const int i0 = ib + lane, i1 = i0 + 32;
                const double x0 = ws.pc[min(i0, FTP - 1)], x1 = ws.pc[min(i1, FTP - 1)];
                const double ta0 = x0 - R, ta1 = x1 - R, tb0 = fmin(x0 + R, Tchi - x0), tb1 = fmin(x1 + R, Tchi - x1);
                int a0 = 0, b0 = 0, a1 = 0, b1 = 0;          // first j with qc[j] > ta / qc[j] >= tb
#pragma unroll
                for (int st = (WS::T < 128 ? 64 : 128); st > 0; st >>= 1) {
                    const double va0 = qc[min(a0 + st - 1, mq)], vb0 = qc[min(b0 + st - 1, mq)];
                    const double va1 = qc[min(a1 + st - 1, mq)], vb1 = qc[min(b1 + st - 1, mq)];
                    a0 += (va0 > ta0) ? 0 : st; b0 += (vb0 >= tb0) ? 0 : st;
                    a1 += (va1 > ta1) ? 0 : st; b1 += (vb1 >= tb1) ? 0 : st;
                }
                if (i0 < mp) { ws.jlo[i0] = (unsigned char)a0; ws.jhi[i0] = (unsigned char)max(a0, b0); }
                if (i1 < mp) { ws.jlo[i1] = (unsigned char)a1; ws.jhi[i1] = (unsigned char)max(a1, b1); }
            }
            __syncwarp();
            // walk FROWS rows at a time over exactly the diagonals those rows need
            for (int i0 = 0; i0 < mp; i0 += FROWS) {
                const int i = i0 + lane;
                int dlo = 1 << 20, dhi = -(1 << 20), r0 = 1 << 20, r1 = -1;
                if (lane < FROWS && i < mp) {
                    const int jl = ws.jlo[i], jh = ws.jhi[i];
                    if (jh > jl) { dlo = jl - i; dhi = jh - 1 - i; r0 = i; r1 = i; }
                }
                dlo = __reduce_min_sync(0xffffffffu, dlo); dhi = __reduce_max_sync(0xffffffffu, dhi);
                r0 = __reduce_min_sync(0xffffffffu, r0); r1 = __reduce_max_sync(0xffffffffu, r1);
                if (r1 >= r0) xi_walk_any<POW2, CHECK>(ws, sw_base, n_base, i0, r0, r1, mq, dlo, dhi, bp, g, (unsigned)c0, np1, lane, evaluated, conflicts, ds);
            }
        }
    }
    if (win_c0 >= 0) xi_merge(ws, P, win_c0, win_reg, lane);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
    if (lane == 0 && evaluated) atomicAdd(&P.counters[2], evaluated);
    if (CHECK) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) conflicts += __shfl_xor_sync(0xffffffffu, conflicts, o);
        if (lane == 0 && conflicts) atomicAdd(&P.counters[5], (unsigned long long)conflicts);
    }
}

}  // namespace

namespace {
__global__ void k_check_region(const int32_t *region, int64_t n, int n_region, unsigned long long *flag)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p < n && (unsigned)region[p] >= (unsigned)n_region) atomicMax(flag, 1ull);
}
}  // namespace

// region == NULL: eq. 2.4 over the whole list.  Otherwise (NEXT-1) one set of accumulators per sub-sample.
static lya_status xi_run(lya_ctx *ctx, const lya_plan *pl, const int32_t *region, int n_region,
                         double *S, double *W, uint64_t *N, double *xi, lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pl) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf: plan is NULL");
    if (!pl->has_xi) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf: the plan was created without want_xi");
    LYA_CUDA(lya_enter(ctx));
    const lya_forests *f = &pl->f;
    const lya_binning *b = &pl->b;
    const int nb = b->n_par * b->n_perp;
    const int n_reg = region ? n_region : 1;
    const size_t nbt = (size_t)nb * n_reg;                     // accumulator entries
    cudaStream_t s = ctx->stream;
    const BinParams bp = pl->bp;
    if (region) {
        if (n_region < 1 || (int64_t)n_region * nb > ((int64_t)1 << 28))
            return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi2pcf_sub: need 1 <= n_region and n_region * bins <= 2^28");
        cudaMemsetAsync(ctx->d_counters + 12, 0, sizeof(unsigned long long), s);
        if (f->n_forest > 0)
            { k_check_region<<<(unsigned)((f->n_forest + 255) / 256), 256, 0, s>>>(region, f->n_forest, n_region, ctx->d_counters + 12); lya_note_launch(); }
        unsigned long long bad = 0;
        LYA_CUDA(cudaMemcpyAsync(&bad, ctx->d_counters + 12, sizeof(bad), cudaMemcpyDeviceToHost, s));
        LYA_CUDA(cudaStreamSynchronize(s));
        if (bad) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_sub: region[] must lie in [0, n_region)");
    }
    const bool use_fast = pl->use_fast;
    const LyaBuckets &bk = pl->bk;
    double *acc = NULL;                         // [S | W | N] accumulators
    auto cleanup = [&]() { lya_free(acc); };
    cudaEventRecord(ctx->ev[3], s);
    cudaError_t e = lya_malloc(&acc, nbt * 24);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_malloc(xi accumulators)");
    cudaMemsetAsync(acc, 0, nbt * 24, s);
    cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);

    XiParams P;
    P.pix_off = f->pix_off; P.chi = f->chi; P.w = f->w; P.delta = f->delta;
    P.ux = f->ux; P.uy = f->uy; P.uz = f->uz;
    P.pq = use_fast ? bk.pq + 2 * (bk.n_fast + bk.n_fast2) : pl->pq;
    P.n_pairs = use_fast ? bk.n_long + bk.n_generic : pl->n_pairs;     // (long pairs take the generic xi kernel)
    P.n_forest = f->n_forest;
    P.bp = bp;
    P.S = acc; P.W = acc + nbt; P.N = (unsigned long long *)(acc + 2 * nbt);
    P.counters = ctx->d_counters;

    cudaEventRecord(ctx->ev[0], s);
    if (use_fast && bk.n_fast + bk.n_fast2 > 0) {
        XiFastParams F;
        F.prep = pl->prep; F.pq = bk.pq; F.n_pairs = bk.n_fast; F.bp = bp;
        F.S = P.S; F.W = P.W; F.N = P.N; F.counters = ctx->d_counters;
        F.region = region; F.n_region = n_reg;
        F.merge_every = ctx->xi_merge_every;
        const int fgrid = ctx->sm_count;
        auto launch = [&](auto kern, size_t fsmem, int threads) {
            cudaError_t le = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem);
            if (le == cudaSuccess) { kern<<<fgrid, threads, fsmem, s>>>(F); lya_note_launch(); }
            return le;
        };
        if (bk.n_fast > 0) {                                   // class 0
            const size_t fsmem = sizeof(FastWarp) * FW;
            if (ctx->check_holders) e = bp.pow2 ? launch(k_xi_fast<true, true, 0>, fsmem, FTHREADS) : launch(k_xi_fast<false, true, 0>, fsmem, FTHREADS);
            else e = bp.pow2 ? launch(k_xi_fast<true, false, 0>, fsmem, FTHREADS) : launch(k_xi_fast<false, false, 0>, fsmem, FTHREADS);
            if (e == cudaSuccess) e = cudaGetLastError();
            if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi_fast launch"); }
        }
        if (bk.n_fast2 > 0) {                                  // class 1: its own range of the bucketed list, its own chunk counter
            F.pq = bk.pq + 2 * bk.n_fast; F.n_pairs = bk.n_fast2;
            cudaMemsetAsync(ctx->d_counters + 4, 0, sizeof(unsigned long long), s);
            const size_t fsmem = sizeof(FastWarpT<XiCfg<1>::T>) * XiCfg<1>::WARPS;
            const int threads = XiCfg<1>::WARPS * 32;
            if (ctx->check_holders) e = bp.pow2 ? launch(k_xi_fast<true, true, 1>, fsmem, threads) : launch(k_xi_fast<false, true, 1>, fsmem, threads);
            else e = bp.pow2 ? launch(k_xi_fast<true, false, 1>, fsmem, threads) : launch(k_xi_fast<false, false, 1>, fsmem, threads);
            if (e == cudaSuccess) e = cudaGetLastError();
            if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi_fast (class 1) launch"); }
        }
    }
    const size_t smem = (((size_t)nb * 20 + 15) & ~(size_t)15) + sizeof(WarpSmem) * XI_WARPS;
    const int grid = ctx->sm_count * 2;
    const int64_t n_chunks = (P.n_pairs + CHUNK - 1) / CHUNK;
    int launches = 0;
    unsigned long long h[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (region && P.n_pairs > 0) {                 // sub-sample mode: the block-level histogram of k_xi cannot be used
        const int dgrid = (int)((P.n_pairs + 7) / 8 < (int64_t)ctx->sm_count * 8 ? (P.n_pairs + 7) / 8 : (int64_t)ctx->sm_count * 8);
        if (bp.pow2) { k_xi_direct<true><<<dgrid, 256, 0, s>>>(P, region); lya_note_launch(); }
        else { k_xi_direct<false><<<dgrid, 256, 0, s>>>(P, region); lya_note_launch(); }
        e = cudaGetLastError();
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi_direct launch"); }
    }
    while (!region && P.n_pairs > 0) {
        switch (ctx->generic_diagonals) {
        case 1: e = launch_xi<1>(P, grid, smem, s); break;
        case 4: e = launch_xi<4>(P, grid, smem, s); break;
        default: e = launch_xi<2>(P, grid, smem, s); break;
        }
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi launch"); }
        ++launches;
        e = cudaMemcpyAsync(h, ctx->d_counters, 4 * sizeof(h[0]), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "k_xi"); }
        if ((int64_t)h[0] >= n_chunks) break;      // every chunk claimed (warps stop at their u32 budget)
        if (launches > 100000) { cleanup(); return lya_fail(ctx, LYA_ERR_CUDA, "k_xi made no progress"); }
    }
    cudaEventRecord(ctx->ev[1], s);
    { k_xi_finalize<<<(unsigned)((nbt + 255) / 256), 256, 0, s>>>(P.S, P.W, P.N, (int)nbt, S, W, (unsigned long long *)N, xi); lya_note_launch(); }
    cudaEventRecord(ctx->ev[2], s);
    e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cleanup(); return lya_cuda_fail(ctx, e, "lya_xi2pcf"); }
    if (h[3] != 0) { cleanup(); return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)"); }
    if (h[5] != 0) { cleanup(); return lya_fail(ctx, LYA_ERR_CUDA, "k_xi_fast: %llu sub-histogram entries had two holders (LYA_OPT_CHECK_HOLDERS)", h[5]); }
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_forest_pairs = (uint64_t)pl->n_pairs;
        stats->n_visited = use_fast ? pl->visited : h[1];
        stats->n_evaluated = h[2];
        // n_binned = sum N: small D2H
        unsigned long long *hN = (unsigned long long *)malloc(sizeof(unsigned long long) * nbt);
        if (hN && cudaMemcpy(hN, P.N, sizeof(unsigned long long) * nbt, cudaMemcpyDeviceToHost) == cudaSuccess)
            for (size_t k = 0; k < nbt; ++k) stats->n_binned += hN[k];
        free(hN);
        cudaEventElapsedTime(&stats->ms_main, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&stats->ms_total, ctx->ev[3], ctx->ev[2]);
    }
    cleanup();
    return LYA_OK;
}

extern "C" lya_status lya_xi2pcf_plan(lya_ctx *ctx, const lya_plan *plan,
                                      double *S, double *W, uint64_t *N, double *xi, lya_stats *stats)
{
    return xi_run(ctx, plan, NULL, 1, S, W, N, xi, stats);
}

extern "C" lya_status lya_xi2pcf(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                                 double *S, double *W, uint64_t *N, double *xi, lya_stats *stats)
{
    lya_plan *pl = NULL;
    lya_status st = lya_plan_create(ctx, f, b, pairs, 1, 0, &pl);
    if (st) return st;
    st = xi_run(ctx, pl, NULL, 1, S, W, N, xi, stats);
    lya_plan_free(ctx, pl);
    return st;
}

extern "C" lya_status lya_xi2pcf_sub(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                                     const int32_t *region, int32_t n_region,
                                     double *S, double *W, uint64_t *N, lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!region) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_sub: region is NULL");
    lya_plan *pl = NULL;
    lya_status st = lya_plan_create(ctx, f, b, pairs, 1, 0, &pl);
    if (st) return st;
    st = xi_run(ctx, pl, region, n_region, S, W, N, NULL, stats);
    lya_plan_free(ctx, pl);
    return st;
}

// ======================= NEXT-1, second half: weighted sums of r_par, r_perp, z per bin ==================
// Rpar_A = sum om r_par, Rperp_A = sum om r_perp, Z_A = sum om (z_i + z_j) / 2, W_A = sum om over the in-grid
// pixel pairs of bin A, om = w_i w_j (the PICCA-like table carries the weighted mean
// coordinates of every bin; the means are these sums over W_A).  A second, cheap mode next to the pair kernel:
// one warp per forest pair, lanes over the pixel pairs, block-level shared histogram (fp64 shared atomics are a
// CAS loop here -- acceptable for an output computed once per analysis), merged with global fp64 atomics.
namespace {
constexpr int MEAN_THREADS = 256;
template <bool POW2>
__global__ void __launch_bounds__(MEAN_THREADS) k_xi_means(XiParams P, const double *z, double *out /* [4][nb] */)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const BinParams bp = P.bp;
    const int nb = bp.n_par * bp.n_perp;
    double *h = (double *)smem_raw;                                   // [4][nb]
    for (int k = threadIdx.x; k < 4 * nb; k += MEAN_THREADS) h[k] = 0.0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t k = warp; k < P.n_pairs; k += n_warps) {
        const int p = P.pq[2 * k], q = P.pq[2 * k + 1];
        if ((unsigned)p >= (unsigned)P.n_forest || (unsigned)q >= (unsigned)P.n_forest) {
            if (lane == 0) atomicMax(&P.counters[3], (unsigned long long)LYA_DEV_BAD_PAIR);
            continue;
        }
        const int64_t op = P.pix_off[p], oq = P.pix_off[q];
        const int np = (int)(P.pix_off[p + 1] - op), nq = (int)(P.pix_off[q + 1] - oq);
        if (np == 0 || nq == 0) continue;
        double s, c;
        lya_pair_sc(P.ux[p], P.uy[p], P.uz[p], P.ux[q], P.uy[q], P.uz[q], s, c);
        const PairBin g = lya_make_pairbin(bp, s, c);
        int i = 0, j = lane;                                           // lanes over the pixel pairs, row-major
        while (j >= nq) { j -= nq; ++i; }
        while (i < np) {
            const double ci = P.chi[op + i], cj = P.chi[oq + j];
            const int A = lya_pix_bin<POW2>(bp, g, ci, cj);
            if (A >= 0) {
                const double om = P.w[op + i] * P.w[oq + j];
                const double rpar = __dmul_rn(fabs(__dsub_rn(ci, cj)), g.c), rperp = __dmul_rn(__dadd_rn(ci, cj), g.s);
                atomicAdd(&h[A], om * rpar);
                atomicAdd(&h[nb + A], om * rperp);
                atomicAdd(&h[2 * nb + A], om * (0.5 * (z[op + i] + z[oq + j])));
                atomicAdd(&h[3 * nb + A], om);
            }
            j += 32;
            while (j >= nq) { j -= nq; ++i; }
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < 4 * nb; k += MEAN_THREADS)
        if (h[k] != 0.0) atomicAdd(&out[k], h[k]);
}
}  // namespace

extern "C" lya_status lya_xi2pcf_means(lya_ctx *ctx, const lya_forests *f, const lya_binning *b, const lya_pairs *pairs,
                                       const double *z, double *Rpar, double *Rperp, double *Z, double *W)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pairs || !Rpar || !Rperp || !Z) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_means: NULL argument");
    lya_status st = lya_check_binning(ctx, b);
    if (st) return st;
    st = lya_check_forests_host(ctx, f, true, false, false);
    if (st) return st;
    if (f->n_forest > 0 && !(f->ux && f->uy && f->uz)) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_means needs ux,uy,uz (device)");
    if (f->n_pix > 0 && !z) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_means: z is NULL");
    LYA_CUDA(lya_enter(ctx));
    st = lya_validate_forests(ctx, f, false, false, NULL);
    if (st) return st;
    const int nb = b->n_par * b->n_perp;
    cudaStream_t s = ctx->stream;
    double *acc = NULL;
    LYA_CUDA(lya_malloc(&acc, sizeof(double) * 4 * (size_t)nb));
    cudaMemsetAsync(acc, 0, sizeof(double) * 4 * (size_t)nb, s);
    cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
    XiParams P;
    memset(&P, 0, sizeof(P));
    P.pix_off = f->pix_off; P.chi = f->chi; P.w = f->w; P.delta = NULL;
    P.ux = f->ux; P.uy = f->uy; P.uz = f->uz;
    P.pq = pairs->pq; P.n_pairs = pairs->n; P.n_forest = f->n_forest;
    P.bp = lya_make_binparams(b);
    P.counters = ctx->d_counters;
    cudaError_t e = cudaSuccess;
    if (pairs->n > 0) {
        const size_t smem = sizeof(double) * 4 * (size_t)nb;
        const int64_t want = (pairs->n + 7) / 8;
        const int grid = (int)(want < (int64_t)ctx->sm_count * 2 ? want : (int64_t)ctx->sm_count * 2);
        if (P.bp.pow2) {
            e = cudaFuncSetAttribute(k_xi_means<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) { k_xi_means<true><<<grid, MEAN_THREADS, smem, s>>>(P, z, acc); lya_note_launch(); }
        } else {
            e = cudaFuncSetAttribute(k_xi_means<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess) { k_xi_means<false><<<grid, MEAN_THREADS, smem, s>>>(P, z, acc); lya_note_launch(); }
        }
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    const size_t bytes = sizeof(double) * (size_t)nb;
    if (e == cudaSuccess) e = cudaMemcpyAsync(Rpar, acc, bytes, cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(Rperp, acc + nb, bytes, cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(Z, acc + 2 * nb, bytes, cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess && W) e = cudaMemcpyAsync(W, acc + 3 * nb, bytes, cudaMemcpyDeviceToDevice, s);
    unsigned long long h[4] = {0, 0, 0, 0};
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    lya_free(acc);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_xi2pcf_means");
    if (h[3] != 0) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
    return LYA_OK;
}

// xi_A = S_A / W_A (0 where W_A == 0) from already-summed numerators (section 8(e): after the all-reduce).
extern "C" lya_status lya_xi_normalise(lya_ctx *ctx, int64_t n, const double *S, const double *W, double *xi)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (n < 0 || (n > 0 && (!S || !W || !xi))) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi_normalise: bad arguments");
    if (n > ((int64_t)1 << 30)) return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi_normalise: n above 2^30");
    LYA_CUDA(lya_enter(ctx));
    if (n > 0) {
        { k_xi_finalize<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(S, W, NULL, (int)n, NULL, NULL, NULL, xi); lya_note_launch(); }
        LYA_CUDA(cudaGetLastError());
    }
    return LYA_OK;
}

// ======================= lya_xi2pcf_plan_noalloc: stage 2 on a plan, allocating nothing ==================
// For callers that cannot allocate device memory in the call (CUDA graph capture around it is not what is meant --
// the call synchronises; but serving loops and harnesses that forbid cudaMalloc): the same kernels as
// lya_xi2pcf_plan, with the [S | W | N] accumulators -- the one piece of scratch memory stage 2 needs -- in a
// file-scope device array instead of a stream-ordered allocation.  The array is part of the library image: every
// GPU that loads liblya.so holds LYA_XI_NOALLOC_MAX_BINS * 24 bytes (60 KB) until the process exits.
// In HOST code the array's name is a host-side stand-in, not a device address, so the address is asked for once
// per device (that device current) with cudaGetSymbolAddress and handed to the kernels as an ordinary pointer.
// Every call on a device shares the array and finds the last call's sums in it: it is cleared on the ctx stream
// first, and calls that overlap on the GPU (two contexts / streams of one device) RACE -- see include/lya.h.
static __device__ __align__(256) double g_xi_noalloc_acc[3 * LYA_XI_NOALLOC_MAX_BINS];

namespace {
constexpr int XI_NOALLOC_MAX_DEVICES = 64;
double *g_xi_noalloc_ptr[XI_NOALLOC_MAX_DEVICES];      // device address of g_xi_noalloc_acc, per device ordinal (0 = not asked yet)
}  // namespace

extern "C" lya_status lya_xi2pcf_plan_noalloc(lya_ctx *ctx, const lya_plan *pl,
                                              double *S, double *W, uint64_t *N, double *xi, lya_stats *stats)
{
    if (!ctx) return LYA_ERR_INVALID_ARG;
    if (!pl) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_plan_noalloc: plan is NULL");
    if (!pl->has_xi) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_plan_noalloc: the plan was created without want_xi");
    if (!S || !W || !N || !xi) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "lya_xi2pcf_plan_noalloc: S, W, N and xi are all required");
    const lya_forests *f = &pl->f;
    const int nb = pl->b.n_par * pl->b.n_perp;
    if (nb > LYA_XI_NOALLOC_MAX_BINS)
        return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi2pcf_plan_noalloc: %d bins, the static accumulators hold at most %d "
                        "(use lya_xi2pcf_plan)", nb, LYA_XI_NOALLOC_MAX_BINS);
    if (ctx->device < 0 || ctx->device >= XI_NOALLOC_MAX_DEVICES)
        return lya_fail(ctx, LYA_ERR_CAPACITY, "lya_xi2pcf_plan_noalloc: device ordinal %d outside [0, %d)", ctx->device, XI_NOALLOC_MAX_DEVICES);
    LYA_CUDA(lya_enter(ctx));                                      // makes ctx->device current
    if (!g_xi_noalloc_ptr[ctx->device]) {                          // set-up, once per device
        double *ptr = NULL;
        cudaError_t ge = cudaGetSymbolAddress((void **)&ptr, g_xi_noalloc_acc);
        if (ge != cudaSuccess || !ptr) return lya_cuda_fail(ctx, ge, "cudaGetSymbolAddress(g_xi_noalloc_acc)");
        g_xi_noalloc_ptr[ctx->device] = ptr;
    }
    double *acc = g_xi_noalloc_ptr[ctx->device];
    cudaStream_t s = ctx->stream;
    const BinParams bp = pl->bp;
    const bool use_fast = pl->use_fast;
    const LyaBuckets &bk = pl->bk;
    cudaEventRecord(ctx->ev[3], s);
    cudaError_t e = cudaMemsetAsync(acc, 0, (size_t)nb * 24, s);   // the array keeps the last call's sums
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->d_counters, 0, 8 * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_xi2pcf_plan_noalloc: clearing the accumulators");

    XiParams P;
    P.pix_off = f->pix_off; P.chi = f->chi; P.w = f->w; P.delta = f->delta;
    P.ux = f->ux; P.uy = f->uy; P.uz = f->uz;
    P.pq = use_fast ? bk.pq + 2 * bk.n_fast : pl->pq;
    P.n_pairs = use_fast ? bk.n_fast2 + bk.n_long + bk.n_generic : pl->n_pairs;
    P.n_forest = f->n_forest;
    P.bp = bp;
    P.S = acc; P.W = acc + nb; P.N = (unsigned long long *)(acc + 2 * nb);
    P.counters = ctx->d_counters;

    cudaEventRecord(ctx->ev[0], s);
    if (use_fast && bk.n_fast > 0) {
        XiFastParams F;
        F.prep = pl->prep; F.pq = bk.pq; F.n_pairs = bk.n_fast; F.bp = bp;
        F.S = P.S; F.W = P.W; F.N = P.N; F.counters = ctx->d_counters;
        F.region = NULL; F.n_region = 1;
        F.merge_every = ctx->xi_merge_every;
        const size_t fsmem = sizeof(FastWarp) * FW;
        const int fgrid = ctx->sm_count;
        auto launch = [&](auto kern) {
            cudaError_t le = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem);
            if (le == cudaSuccess) { kern<<<fgrid, FTHREADS, fsmem, s>>>(F); lya_note_launch(); }
            return le;
        };
        if (ctx->check_holders) e = bp.pow2 ? launch(k_xi_fast<true, true>) : launch(k_xi_fast<false, true>);
        else e = bp.pow2 ? launch(k_xi_fast<true, false>) : launch(k_xi_fast<false, false>);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "k_xi_fast launch");
    }
    const size_t smem = (((size_t)nb * 20 + 15) & ~(size_t)15) + sizeof(WarpSmem) * XI_WARPS;
    const int grid = ctx->sm_count * 2;
    const int64_t n_chunks = (P.n_pairs + CHUNK - 1) / CHUNK;
    int launches = 0;
    unsigned long long h[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    while (P.n_pairs > 0) {                                        // generic kernel for the rest of the list
        switch (ctx->generic_diagonals) {
        case 1: e = launch_xi<1>(P, grid, smem, s); break;
        case 4: e = launch_xi<4>(P, grid, smem, s); break;
        default: e = launch_xi<2>(P, grid, smem, s); break;
        }
        if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "k_xi launch");
        ++launches;
        e = cudaMemcpyAsync(h, ctx->d_counters, 4 * sizeof(h[0]), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "k_xi");
        if ((int64_t)h[0] >= n_chunks) break;                      // every chunk claimed (warps stop at their u32 budget)
        if (launches > 100000) return lya_fail(ctx, LYA_ERR_CUDA, "k_xi made no progress");
    }
    cudaEventRecord(ctx->ev[1], s);
    { k_xi_finalize<<<(unsigned)((nb + 255) / 256), 256, 0, s>>>(P.S, P.W, P.N, nb, S, W, (unsigned long long *)N, xi); lya_note_launch(); }
    cudaEventRecord(ctx->ev[2], s);
    e = cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return lya_cuda_fail(ctx, e, "lya_xi2pcf_plan_noalloc");
    if (h[3] != 0) return lya_fail(ctx, LYA_ERR_INVALID_ARG, "pair list refers to a forest outside [0, n_forest)");
    if (h[5] != 0) return lya_fail(ctx, LYA_ERR_CUDA, "k_xi_fast: %llu sub-histogram entries had two holders (LYA_OPT_CHECK_HOLDERS)", h[5]);
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        stats->n_forest_pairs = (uint64_t)pl->n_pairs;
        stats->n_visited = use_fast ? pl->visited : h[1];
        stats->n_evaluated = h[2];
        unsigned long long hN[LYA_XI_NOALLOC_MAX_BINS];            // n_binned = sum N (host stack, no allocation)
        if (cudaMemcpy(hN, P.N, sizeof(unsigned long long) * (size_t)nb, cudaMemcpyDeviceToHost) == cudaSuccess)
            for (int k = 0; k < nb; ++k) stats->n_binned += hN[k];
        cudaEventElapsedTime(&stats->ms_main, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&stats->ms_total, ctx->ev[3], ctx->ev[2]);
    }
    return LYA_OK;
}
