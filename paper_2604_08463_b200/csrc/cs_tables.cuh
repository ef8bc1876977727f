// cs_tables.cuh -- the small kernels around the fused ones.
//
//   k_tables    a1  SED factor tables, fp64 math -> fp32 rows                     (Eq. 2)
//   k_merge     a3  second level: fixed-order sum of per-tile partials onto clusters and regions
//   k_cmbvar    f1  variance of the CMB map from the region-reduced sums          (Eq. 10)
//   k_relayout      gathers a data set into the sorted layout of one configuration (cs_internal.h), once per
//                   (configuration, data set) pair of a batch
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"

namespace cs {

// ----------------------------------------------------------------------------------------------------------
// a1: SED factor tables.  One thread per (entry, parameter, band quad).  fp64 -> fp32.
// ----------------------------------------------------------------------------------------------------------
// exp(y) in fp64 for the power-law rows: y = k ln2 + r, |r| <= ln2/2, degree-11 Taylor polynomial (truncation
// 6e-15 relative, far below the fp32 rounding of the stored value), scaled by 2^k through the exponent field.
// k comes from the 1.5 * 2^52 shift (no FRND / F2I on the conversion pipe), the coefficients from the constant bank
// (as 64-bit immediates every one costs two UMOV per use: the kernel is bound by instruction issue), and 2^k is an
// integer add on the high word of the polynomial's value (it lies in [0.7, 1.42] and the result is a normal number).
// Arguments outside the range where 2^k is a normal number give +inf / 0 / NaN by selection (what the library routine
// returns there once rounded to fp32), so that the four values of a thread stay free of branches and interleave.
__constant__ double EXP_C[12] = {1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0, 1.0 / 40320.0, 1.0 / 5040.0, 1.0 / 720.0,
                                 1.0 / 120.0,      1.0 / 24.0,      1.0 / 6.0,      0.5,          1.0,          1.0};
__constant__ double EXP_R[4] = {1.4426950408889634074, 6755399441055744.0, 6.93147180369123816490e-01, 1.90821492927058770002e-10};
__device__ __forceinline__ double exp_pow(double y) {
    const bool ok = fabs(y) < 700.0;               // false for NaN
    const double ys = ok ? y : 0.0;
    const double t = fma(ys, EXP_R[0], EXP_R[1]);  // the integer nearest to y / ln2 sits in the low word
    const double kf = t - EXP_R[1];
    const int k = __double2loint(t);
    double r = fma(-kf, EXP_R[2], ys);
    r = fma(-kf, EXP_R[3], r);
    double p = EXP_C[0];
#pragma unroll
    for (int i = 1; i < 12; ++i) p = fma(p, r, EXP_C[i]);
    const double res = __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
    const double out_of_range = (y > 0.0) ? CUDART_INF : ((y < 0.0) ? 0.0 : y + y);
    return ok ? res : out_of_range;
}

// One value of a power-law row, band constant folded in: c (nu/nu0)^beta = c exp(beta ln(nu/nu0)), rounded to fp32.
// k_tables' form.  (The direct kernel's per-pixel beta_d path, CfgDev::pixbeta, uses powerlaw_pair_f32 below instead: not
// the same bits.)
__device__ __forceinline__ float powerlaw_value(double c, double lnr, double beta) {
    return (float)__dmul_rn(c, exp_pow(__dmul_rn(beta, lnr)));
}

// The same value for two pixels at once in fp32, for the direct kernel's per-pixel beta_d path (CfgDev::pixbeta):
// c 2^(beta L), L = log2(nu/nu0), with beta and L as float pairs (hi, lo) so that the exponent beta L is known to 1e-14:
// p = bh Lh (rounded), e = fma(bh, Lh, -p) (its error, exact), s = e + bh Ll + bl Lh; k = rint(p); r = (p - k) + s with
// |r| <= 1/2; 2^r by MUFU.EX2 (at most two units in the last place), 2^k through the exponent field (k clamped to the
// normal range: beyond it the fp32 table value would be 0 or inf as well).  Relative error <= 2.5e-7 (the table rows
// are correctly rounded, 6e-8); the fp64 expression above costs the direct kernel, which has eight consumer warps per
// SM to fill the fp64 pipe with, more than it saves (measured: DESIGN.md section 7).
__device__ __forceinline__ float2 powerlaw_pair_f32(float ch, float Lh, float Ll, float2 bh, float2 bl) {
    const float2 p = __fmul2_rn(bh, make_float2(Lh, Lh));
    const float2 e = __ffma2_rn(bh, make_float2(Lh, Lh), make_float2(-p.x, -p.y));
    const float2 s = __ffma2_rn(bh, make_float2(Ll, Ll), __ffma2_rn(bl, make_float2(Lh, Lh), e));
    const float2 magic = make_float2(12582912.f, 12582912.f);
    const float2 t = __fadd2_rn(p, magic);
    const float2 kf = __fadd2_rn(t, make_float2(-12582912.f, -12582912.f));
    const float2 r = __fadd2_rn(__fadd2_rn(p, make_float2(-kf.x, -kf.y)), s);
    float ex, ey;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex) : "f"(r.x));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ey) : "f"(r.y));
    const int kx = min(max((int)kf.x, -126), 127), ky = min(max((int)kf.y, -126), 127);
    const float2 sc = make_float2(__int_as_float((kx + 127) << 23), __int_as_float((ky + 127) << 23));
    return __fmul2_rn(__fmul2_rn(make_float2(ch, ch), sc), make_float2(ex, ey));
}

// 1/a for a normal positive double: MUFU.RCP64H seed (about 20 bits) and two Newton steps (error ~1 ulp, no slow path).
__device__ __forceinline__ double rcp_pos(double a) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
    double e = fma(-a, r, 1.0);
    r = fma(r, e, r);
    e = fma(-a, r, 1.0);
    return fma(r, e, r);
}
// expm1(x): for x >= 1/32 the subtraction exp(x) - 1 loses at most five bits of the 6e-15 of exp_pow; smaller (and
// non-positive or non-finite) arguments take the library routine.
__device__ __forceinline__ double expm1_pos(double x) { return (x >= 0.03125 && x < 700.0) ? exp_pow(x) - 1.0 : expm1(x); }

// One block of k_tables' work: TAB_ROWS_PER_BLOCK consecutive parameters from j0 on of entry e, in one aligned 48-byte record
// (no chain of dependent loads through the configuration table, and no block without work).
struct TabBlock {
    int64_t param_off;   // first parameter of the entry
    int64_t tab_row;     // first table row of the entry
    int32_t K0, K1, ktot, j0;
    int32_t e, pixbeta, pad[2];   // pixbeta: the beta_d rows of this entry are not built (CfgDev::pixbeta)
};
constexpr int TAB_SUB = 4;                       // parameters per thread quad
constexpr int TAB_ROWS_PER_BLOCK = 64 * TAB_SUB;

// One thread per (entry, parameter, band quad): four table values and one 16-byte store.  The band constants come from a
// shared-memory copy (indexed by the thread's quad: a constant-bank read would serialise); the parameter load is issued
// before the copy is staged.  grid = number of 64-parameter blocks of the batch, block = 256.
__global__ void __launch_bounds__(256) k_tables(const double *__restrict__ params, const TabBlock *__restrict__ blocks, float *__restrict__ tab,
                                                int32_t *err, const TConst *__restrict__ tcg, const int32_t *__restrict__ skip) {
    __shared__ TConst tc;
    const int4 *bp = reinterpret_cast<const int4 *>(blocks + blockIdx.x);
    const int4 b0 = __ldg(bp), b1 = __ldg(bp + 1), b2 = __ldg(bp + 2);
    const int64_t param_off = ((int64_t)(uint32_t)b0.y << 32) | (uint32_t)b0.x, tab_row = ((int64_t)(uint32_t)b0.w << 32) | (uint32_t)b0.z;
    const int K0 = b1.x, K1 = b1.y, ktot = b1.z, j0 = b1.w, e = b2.x;
    const bool pixbeta = b2.y != 0;
    if (skip && skip[e] != 0) return;
    const int f0 = (threadIdx.x & 3) * 4;
    // the block's TAB_SUB x 64 parameters: all loads first (one latency for the block), then the rows one after the other
    double xs[TAB_SUB];
#pragma unroll
    for (int u = 0; u < TAB_SUB; ++u) {
        const int j = j0 + 64 * u + (threadIdx.x >> 2);
        xs[u] = (j < ktot) ? __ldg(params + param_off + j) : 1.0;
    }
    if (pixbeta && j0 + TAB_ROWS_PER_BLOCK <= K0) {   // block-uniform: beta_d rows the direct kernel evaluates per pixel;
        bool nonfinite = false;                       // nothing to build, only the domain check
#pragma unroll
        for (int u = 0; u < TAB_SUB; ++u) nonfinite = nonfinite || !isfinite(xs[u]);
        if (nonfinite && f0 == 0) atomicOr(err, ERR_DOMAIN);
        return;
    }
    static_assert(sizeof(TConst) / 8 <= 256, "one word per thread");
    if (threadIdx.x < (int)(sizeof(TConst) / 8)) reinterpret_cast<double *>(&tc)[threadIdx.x] = __ldg(reinterpret_cast<const double *>(tcg) + threadIdx.x);
    __syncthreads();
    const int nfreq = tc.nfreq;
    float *row0 = tab + tab_row * NROW;
    bool bad = false;
#pragma unroll
    for (int u = 0; u < TAB_SUB; ++u) {
    const int j = j0 + 64 * u + (threadIdx.x >> 2);
    if (j >= ktot) break;
    const double x = xs[u];
    bad = bad || !isfinite(x);
    float v[4];
    if (j < K0) {
        if (pixbeta) continue;   // evaluated per pixel by the direct kernel
        // dust power-law factor with the band constant folded in: cd[f] * (nu_f/nu0d)^beta_d
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = (f0 + i < nfreq) ? powerlaw_value(tc.cd[f0 + i], tc.lnd[f0 + i], x) : 0.f;
        *reinterpret_cast<float4 *>(row0 + (int64_t)j * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
    } else if (j < K0 + K1) {
        // Planck ratio G = expm1(x0)/expm1(x) and d ln G / dT = (1/T) [ h(x) - h(x0) ],
        // h(x) = x / (1 - e^-x) = x + x / expm1(x): one expm1 and one reciprocal per band
        bad = bad || !(x > 0.0);
        const int k = j - K0;
        float dg[4];
        const double inv_t = 1.0 / x;
        const double x0 = tc.hk * tc.nu0d * inv_t, e0 = expm1_pos(x0), h0 = fma(x0, rcp_pos(e0), x0);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[i] = 0.f; dg[i] = 0.f;
            if (f0 + i < nfreq) {
                const double xf = tc.hk * tc.nu[f0 + i] * inv_t;
                const double re = rcp_pos(expm1_pos(xf));
                v[i] = (float)(e0 * re);
                dg[i] = (float)((fma(xf, re, xf) - h0) * inv_t);
            }
        }
        *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + k) * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
        *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + K1 + k) * NROW + f0) = make_float4(dg[0], dg[1], dg[2], dg[3]);
    } else {
        const int k = j - K0 - K1;
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = (f0 + i < nfreq) ? powerlaw_value(tc.cs[f0 + i], tc.lns[f0 + i], x) : 0.f;
        *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + 2 * K1 + k) * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
    }
    }
    if (bad && f0 == 0) atomicOr(err, ERR_DOMAIN);
}

// ----------------------------------------------------------------------------------------------------------
// a3 second level: grad[e][j] / nll[e][r] = fixed-order (ascending tile) sum over the segments of cluster j / region r,
// which are contiguous in the partial row.
// want_grad = 0: only the region outputs.
// ----------------------------------------------------------------------------------------------------------
// Cluster outputs with at most MERGE_LONG slots (nearly all): one thread each, slots added in ascending order.  Longer
// ranges -- the region outputs (sixteen slots per tile: thousands per entry) and the clusters of a map with a handful
// of patches (K = 1 in the clustering scan: one cluster owns every slot of its term) -- are summed by a whole block:
// thread i adds the slots a+i, a+i+256, ... in ascending order, the 32 lane sums of a warp are combined by a fixed
// xor-shuffle tree and the eight warp sums left to right.  Which way a cluster goes depends on its slot count only, and
// all orders are fixed, so the result is bitwise reproducible and independent of the batch.
// (Measured alternatives for the short clusters, both slower on every configuration: eight lanes per cluster -- eight
// times the threads, each with the same chain of pointer loads in front of one or two slots; warp-cooperative sums from
// 16 slots on -- a warp full of T_d clusters then walks them one after the other.  One thread per long range was the
// long pole of the whole kernel: 1536 dependent adds for a K = 1 map, 192 rounds of loads per lane for a region at nside 128.)
// grid = the batch's work list of blocks (host-built: per entry ceil(ktot / 256) cluster blocks when the gradient is wanted,
// then one block per region -- entries of one batch own between 12 and 6000 parameters, a 2-D grid sized for the
// largest left most blocks without work), block = 256.
constexpr int MERGE_LONG = 64;
struct MergeBlock {
    int32_t e;   // entry
    int32_t b;   // >= 0: cluster block (parameters [256 b, 256 b + 256)); < 0: region -(b + 1)
};
__device__ __forceinline__ double merge_block_sum(const double *__restrict__ row, int a, int b, double *wsum) {
    double acc = 0.0;
#pragma unroll 8
    for (int q = a + (int)threadIdx.x; q < b; q += 256) acc += row[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __syncthreads();   // wsum is free again
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    __syncthreads();
    double tot = wsum[0];
#pragma unroll
    for (int i = 1; i < 8; ++i) tot += wsum[i];
    return tot;
}
__global__ void __launch_bounds__(256) k_merge(const double *__restrict__ partial, int64_t PS, const CfgDev *__restrict__ cfgs,
                                               const int32_t *__restrict__ cfg_of, const int64_t *__restrict__ param_off, int32_t nregion,
                                               const MergeBlock *__restrict__ blocks, double *__restrict__ nll, double *__restrict__ grad,
                                               const int32_t *__restrict__ skip) {
    __shared__ double wsum[8];
    __shared__ int32_t s_long[256][3];   // (a, b, offset of the term's block in the row) of this block's long clusters, by thread
    __shared__ int32_t s_who[256], s_nlong;
    const MergeBlock mb = blocks[blockIdx.x];
    const int e = mb.e;
    if (skip && skip[e] != 0) return;
    const CfgDev *c = cfgs + cfg_of[e];
    const double *erow = partial + (int64_t)e * PS;
    if (mb.b >= 0) {
        const int K0 = c->K[0], K1 = c->K[1], ktot = c->ktot;
        if (threadIdx.x == 0) s_nlong = 0;
        __syncthreads();
        const int v = mb.b * 256 + threadIdx.x;
        const int64_t dst0 = param_off[e] + (int64_t)mb.b * 256;
        if (v < ktot) {
            int t, k;
            if (v < K0) { t = 0; k = v; }
            else if (v < K0 + K1) { t = 1; k = v - K0; }
            else { t = 2; k = v - K0 - K1; }
            const int32_t *ksegptr = c->kseg[t];
            const int base = c->segbase[t];
            const int a = __ldg(ksegptr + k), b = __ldg(ksegptr + k + 1);
            if (b - a <= MERGE_LONG) {
                const double *row = erow + base;
                double acc = 0.0;
#pragma unroll 8
                for (int q = a; q < b; ++q) acc += row[q];
                grad[dst0 + threadIdx.x] = acc;
            } else {
                s_long[threadIdx.x][0] = a; s_long[threadIdx.x][1] = b; s_long[threadIdx.x][2] = base;
                s_who[atomicAdd(&s_nlong, 1)] = threadIdx.x;
            }
        }
        __syncthreads();
        const int nlong = s_nlong;
        for (int i = 0; i < nlong; ++i) {   // in any order: every sum is on its own
            const int who = s_who[i];
            const double tot = merge_block_sum(erow + s_long[who][2], s_long[who][0], s_long[who][1], wsum);
            if (threadIdx.x == 0) grad[dst0 + who] = tot;
        }
    } else {
        const int r = -(mb.b + 1);
        const int32_t *ksegptr = c->kseg[3];
        const int a = __ldg(ksegptr + r), b = __ldg(ksegptr + r + 1);
        const double tot = merge_block_sum(erow + c->segbase[3], a, b, wsum);
        if (threadIdx.x == 0) nll[(int64_t)e * nregion + r] = tot;
    }
}

// f1 (Eq. 10): variance of the CMB map per entry and region from the four region-reduced sums.
__global__ void __launch_bounds__(128) k_cmbvar(const double *__restrict__ partial, int64_t PS, const MapDev *__restrict__ maps,
                                                const CfgDev *__restrict__ cfgs, const int32_t *__restrict__ cfg_of,
                                                const int32_t *__restrict__ npix_live, int32_t nregion, int32_t batch,
                                                double *__restrict__ var) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= batch * nregion) return;
    const int e = i / nregion, r = i - e * nregion;
    const MapDev *m = maps + cfgs[cfg_of[e]].map[3];
    const int32_t *ksegptr = m->ksegptr;
    const int32_t nseg = m->nseg;
    double s[4];
    for (int t = 0; t < 4; ++t) {
        const double *row = partial + (int64_t)e * PS + (int64_t)t * nseg;
        double acc = 0.0;
        for (int q = ksegptr[r]; q < ksegptr[r + 1]; ++q) acc += row[q];
        s[t] = acc;
    }
    const double n = (double)npix_live[cfg_of[e] * nregion + r];
    var[i] = n > 0 ? (s[2] / n - (s[0] / n) * (s[0] / n)) + (s[3] / n - (s[1] / n) * (s[1] / n)) : 0.0;
}

// Private copy of one data set in the sorted layout of one configuration: copy[tile (stride job.tstride)][half][row][x] =
// d[data][row][pospix[tile*TPX + half*256 + x]], zero at pad positions.  grid = (ntile, pairs), block = TPX.
struct CopyJob {
    int32_t cfg, data;
    int64_t off;       // float offset of the copy's tile 0 inside dcopy
    int64_t tstride;   // floats from one tile of the copy to the next (see "tile-major" in cs_internal.h)
};
__global__ void __launch_bounds__(TPX) k_relayout(const float *__restrict__ d, int64_t npix, int32_t nrows, const CfgDev *__restrict__ cfgs,
                                                  const CopyJob *__restrict__ jobs, float *__restrict__ dcopy) {
    const CopyJob job = jobs[blockIdx.y];
    const CfgDev *cf = cfgs + job.cfg;
    const int tile = blockIdx.x;
    if (tile >= cf->ntile) return;
    const int x = threadIdx.x;
    const int32_t pix = cf->pospix[(int64_t)tile * TPX + x];
    const float *src = d + (int64_t)job.data * nrows * npix + (pix >= 0 ? pix : 0);
    float *dst = dcopy + job.off + (int64_t)tile * job.tstride + (x >> 8) * nrows * HALF + (x & (HALF - 1));
    for (int r = 0; r < nrows; ++r) dst[r * HALF] = (pix >= 0) ? __ldg(src + (int64_t)r * npix) : 0.f;
}

}  // namespace cs
