// lya_walk.cuh -- device helpers shared by the fast pair kernels (xi2pcf.cu, dmat.cu):
// predicated shared-memory accesses, the per-row window search, the stage-4 mask arithmetic.
// (CUDA path only; the CPU oracle shares nothing with this.)
#pragma once
#include "lya_internal.cuh"

// ---- predicated shared-memory accesses (no divergence in the pair loops) ----------------------
__device__ __forceinline__ void sts_v2_if(bool p, unsigned addr, double x, double y)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %0, 0;\n @q st.shared.v2.f64 [%1], {%2, %3};\n}"
                 :: "r"((unsigned)p), "r"(addr), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void lds_v2_if(bool p, unsigned addr, double &x, double &y)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %2, 0;\n @q ld.shared.v2.f64 {%0, %1}, [%3];\n}"
                 : "+d"(x), "+d"(y) : "r"((unsigned)p), "r"(addr) : "memory");
}
__device__ __forceinline__ void sts_u32_if(bool p, unsigned addr, unsigned v)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %0, 0;\n @q st.shared.u32 [%1], %2;\n}"
                 :: "r"((unsigned)p), "r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void lds_u32_if(bool p, unsigned addr, unsigned &v)
{
    asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %1, 0;\n @q ld.shared.u32 %0, [%2];\n}"
                 : "+r"(v) : "r"((unsigned)p), "r"(addr) : "memory");
}
// plain shared-memory loads by 32-bit shared address (lets the compiler fold immediate offsets)
__device__ __forceinline__ double2 lds_v2(unsigned addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds_f64(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// ---- stage 4: the keep mask (integer only) -------------------------------
__device__ __forceinline__ unsigned long long lya_mix64(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__device__ __forceinline__ unsigned long long lya_key_lo(unsigned long long seed, unsigned long long id)
{
    return lya_mix64(seed + id * 0x9E3779B97F4A7C15ULL);
}
__device__ __forceinline__ unsigned long long lya_key_hi(unsigned long long seed, unsigned long long id)
{
    return lya_mix64((seed ^ 0xD1B54A32D192ED03ULL) + id * 0x9E3779B97F4A7C15ULL);
}
// the pair part on precomputed pixel keys: top 32 bits of the low 64 bits of (x ^ x >> 32) * K
__device__ __forceinline__ unsigned lya_pair_hash32(unsigned long long klo, unsigned long long khi)
{
    const unsigned long long x = klo + khi;
    const unsigned xh = (unsigned)(x >> 32), xl = (unsigned)x ^ xh;
    const unsigned Kl = 0x6659FD93u, Kh = 0xD6E8FEB8u;
    return __umulhi(xl, Kl) + xl * Kh + xh * Kl;
}
__device__ __forceinline__ bool lya_keep_pair(unsigned long long klo, unsigned long long khi, unsigned long long thr)
{
    return (unsigned long long)lya_pair_hash32(klo, khi) >= thr;
}

// ---- per-row windows ---------------------------------------------------------------------------
// in-grid test of one pixel pair (the exact bin arithmetic of lya_pix_bin)
template <bool POW2>
__device__ __forceinline__ bool lya_in_grid(const BinParams &bp, const PairBin &g, double chi_i, double chi_j)
{
    return lya_pix_bin<POW2>(bp, g, chi_i, chi_j) >= 0;
}

// EXACT window of row x = chi_i against the increasing chi of q (shared memory, mq pixels):
// [jlo, jhi) = the q pixels whose pair with i is inside the grid, jx = first j with chi_j > chi_i
// (clamped into [jlo, jhi]).  The in-grid set of a row is contiguous: r_perp grows with j, r_par
// falls towards chi_j = chi_i and grows after it, and every rounded operation is monotone.  Lower-bound
// searches give a conservative superset (margins R, Tchi); the ends are then moved with the exact bin
// test, so that callers can take "j in [jlo, jhi)" for "in the grid" without redoing geometry.
// The three searches run as ONE branch-free loop of fixed trip count (three independent dependency chains in
// flight; as three data-dependent binary searches one after the other they were pure latency).  STEP0: a power of two
// with 2 * STEP0 > the longest q; qce[mq] must be a sentinel (chi far above every real pixel).
template <bool POW2, int STEP0>
__device__ __forceinline__ void lya_row_window_ilp(const BinParams &bp, const PairBin &g, const double2 *qce, int mq,
                                                   double x, double R, double Tchi, int &jlo, int &jx, int &jhi)
{
    const double ta = x - R, tb = fmin(x + R, Tchi - x);
    int a = 0, b = 0, c = 0;                     // first j with chi_j > ta / chi_j >= tb / chi_j > x
#pragma unroll
    for (int s = STEP0; s > 0; s >>= 1) {
        const double va = qce[min(a + s - 1, mq)].x, vb = qce[min(b + s - 1, mq)].x, vc = qce[min(c + s - 1, mq)].x;
        a += (va > ta) ? 0 : s;
        b += (vb >= tb) ? 0 : s;
        c += (vc > x) ? 0 : s;
    }
    jlo = a; jhi = max(b, a);
    while (jlo < jhi && !lya_in_grid<POW2>(bp, g, x, qce[jlo].x)) ++jlo;
    while (jhi > jlo && !lya_in_grid<POW2>(bp, g, x, qce[jhi - 1].x)) --jhi;
    jx = min(max(c, jlo), jhi);
}
