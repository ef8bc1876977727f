// cs_cells.cuh -- f3: the cell-compressed likelihood (PAPER.md:L95 patch model, L80 Eq. 6).
//
// All pixels of a cell (same cluster triple and region) share A, so their contribution to Eq. 6 depends on the data
// only through the cell's second moments:
//
//     sum_{p in cell} sum_S b_S^T M^-1 b_S  =  tr( M^-1 A^T T A ),        T = N^-1 (sum_{p,S} d_S d_S^T) N^-1   [F x F]
//
// T is independent of the parameters: k_cc_moments builds it once per (configuration, data set) pair, in fp64, from
// the pair's private sorted copy of the data.  A likelihood + gradient evaluation then costs one F x F contraction per cell instead of one
// pass over every pixel (k_like_cc, fp64; one thread per (entry, cell)):
//
//     u_i  = T a_i   (a_0 = 1, a_1 = a_d, a_2 = a_s) ;   B = A^T T A ;   nll_cell = -1/2 tr(M^-1 B)
//     g_th = X[j,:] . P_th  -  M^-1[j,:] . (U^T a'_th) ,   X = M^-1 B M^-1 ,  P_th = A^T N^-1 a'_th ,  j = column of th
//
// which is Eq. 17 summed over the cell's pixels with s = M^-1 A^T N^-1 d written out.  The per-cell
// terms are then summed onto clusters and regions in ascending cell order (k_cc_reduce, fp64, deterministic).
// Cells are the tile-cells of the configuration's sorted layout (a cell that straddles a tile boundary counts twice,
// which changes nothing in the sums).  Pays when cells hold more than ~8 pixels (960 B of moments against 120 B per
// pixel); useless at K ~ npix.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"

namespace cs {

constexpr int CC_NMOM = NROW * (NROW - 1) / 2;   // 120 = 15 * 16 / 2 unique entries of a symmetric 15 x 15 (generic nfreq <= 16: 136 would be needed; see CC_MAXF)
#ifndef CS_CC_UNROLL
#define CS_CC_UNROLL 15
#endif
constexpr int CC_UNROLL = CS_CC_UNROLL;           // rows of T in flight per thread in k_like_cc
constexpr int CC_MAXF = 15;                      // f3 is built for nfreq <= 15 (the LiteBIRD-like band set)
__host__ __device__ __forceinline__ int cc_idx(int f, int g) {   // packed upper triangle of a 15 x 15 symmetric matrix, f <= g
    return f * CC_MAXF - (f * (f - 1)) / 2 + (g - f);
}

// Global (per configuration) cell list of the sorted layout.
struct CellsDev {
    const int32_t *cellpos;    // [ncell] first position of the cell (global position index = tile * TPX + offset)
    const int32_t *celllen;    // [ncell] positions it covers (pads included)
    const int32_t *cellrows;   // [ncell][4] table rows (Fd', G, dlnG, Fs') = CfgDev::cellrows
    const int32_t *cellreg;    // [ncell] region
    const int32_t *kptr[4];    // CSR cluster (t = 0..2) / region (t = 3) -> cells: [K_t + 1]
    const int32_t *klist[4];   // [ncell] cells of each cluster in ascending order
    int32_t ncell;
    int32_t pad;
};

struct MomJob {
    int32_t cfg, data;
    int64_t off;        // double offset of the pair's moments [CC_NMOM][ncell] inside the moments buffer
    int64_t copy_off;   // float offset of the pair's private sorted copy inside dcopy
    int64_t tstride;    // floats from one tile of the copy to the next
};

// Second moments of one (configuration, data set) pair: T = N^-1 (D_Q D_Q^T + D_U D_U^T) N^-1 with D_S the [nfreq x pixels]
// block of the cell's data -- a dense contraction over the pixels, the one step of this library that is GEMM-shaped, on
// the fp64 tensor cores (mma.sync m8n8k4: the fp32 data are promoted exactly, products and sums are fp64).
// One warp per cell; the 15 bands are two row blocks of 8 (the 16th row is zero), the pixels go through in steps of 4.
// Lane (r, k) = (lane / 4, lane % 4) holds D[8 b + r][pixel j0 + k] for both row blocks b and both Stokes parameters:
// that register is its A fragment of block b (row r, column k) and, the matrix being D D^T, also its B fragment
// (row k, column r) -- no shared memory and no transposition.  The cell's pixels are consecutive positions of the
// pair's private sorted copy (pads read as zero data), 16 contiguous bytes per row and step.
// Three accumulator tiles (0,0), (0,1), (1,1) of 8 x 8; lane (r, k) ends with the entries (r, 2k) and (r, 2k + 1) of each.
// grid = (ceil(ncell_max / 4), pairs), block = 128.
__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__global__ void __launch_bounds__(128) k_cc_moments(const float *__restrict__ dcopy, int32_t nfreq, const CellsDev *__restrict__ cells,
                                                    const MomJob *__restrict__ jobs, const float *__restrict__ w, double *__restrict__ mom) {
    const MomJob job = jobs[blockIdx.y];
    const CellsDev *cl = cells + job.cfg;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c = blockIdx.x * 4 + warp;
    if (c >= cl->ncell) return;   // whole warps: the cell is the warp's
    const int pos0 = cl->cellpos[c], len = cl->celllen[c];
    const int nrows = 2 * nfreq;
    const float *dd = dcopy + job.copy_off;
    const int r = lane >> 2, k = lane & 3;
    const int f0 = r, f1 = 8 + r;   // the lane's band in the two row blocks
    const bool has0 = f0 < nfreq, has1 = f1 < nfreq;
    double c00[2] = {0.0, 0.0}, c01[2] = {0.0, 0.0}, c11[2] = {0.0, 0.0};
#pragma unroll 2
    for (int j0 = 0; j0 < len; j0 += 4) {
        const int j = j0 + k;
        float q0 = 0.f, u0 = 0.f, q1 = 0.f, u1 = 0.f;
        if (j < len) {
            const int pos = pos0 + j, tile = pos / TPX, within = pos - tile * TPX;
            const float *src = dd + (int64_t)tile * job.tstride + (within / HALF) * nrows * HALF + (within % HALF);
            if (has0) { q0 = __ldg(src + (2 * f0) * HALF); u0 = __ldg(src + (2 * f0 + 1) * HALF); }
            if (has1) { q1 = __ldg(src + (2 * f1) * HALF); u1 = __ldg(src + (2 * f1 + 1) * HALF); }
        }
        const double dq0 = (double)q0, du0 = (double)u0, dq1 = (double)q1, du1 = (double)u1;
        dmma_m8n8k4(c00, dq0, dq0); dmma_m8n8k4(c00, du0, du0);
        dmma_m8n8k4(c01, dq0, dq1); dmma_m8n8k4(c01, du0, du1);
        dmma_m8n8k4(c11, dq1, dq1); dmma_m8n8k4(c11, du1, du1);
    }
    // the unique entries f <= g < 15 (zero where a band is beyond nfreq), weighted by w_f w_g
    const int ncell = cl->ncell;
    double *out = mom + job.off + c;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int g0 = 2 * k + i, g1 = 8 + g0;
        const double wf0 = has0 ? (double)w[f0] : 0.0, wf1 = has1 ? (double)w[f1] : 0.0;
        const double wg0 = (g0 < nfreq) ? (double)w[g0] : 0.0, wg1 = (g1 < nfreq) ? (double)w[g1] : 0.0;
        if (f0 <= g0) out[(int64_t)cc_idx(f0, g0) * ncell] = wf0 * wg0 * c00[i];
        if (g1 < CC_MAXF) out[(int64_t)cc_idx(f0, g1) * ncell] = wf0 * wg1 * c01[i];
        if (f1 < CC_MAXF && g1 < CC_MAXF && f1 <= g1) out[(int64_t)cc_idx(f1, g1) * ncell] = wf1 * wg1 * c11[i];
    }
}

// One (entry, cell): nll term and the three gradient terms from the cell's moments, in fp64.
// grid = (ceil(ncell_max / 128), batch), block = 128.  out[e] = [4][ncell_max] (ll, g_beta_d, g_T_d, g_beta_s).
// Every unique moment T_fg is loaded once (coalesced over the cells of a warp) and used for both rows it belongs to:
// u_i[f] += T_fg a_i[g], u_i[g] += T_fg a_i[f].  The loops are fully unrolled so that u_0, u_1, u_2 and the two
// non-trivial columns of A (75 doubles) stay in registers; the contractions with u come first, the sums that need only
// the columns (M, P) after u is dead, which keeps the kernel below 255 registers without spills.
__global__ void __launch_bounds__(128, 2) k_like_cc(const CfgDev *__restrict__ cfgs, const CellsDev *__restrict__ cells,
                                                    const int32_t *__restrict__ cfg_of, const int64_t *__restrict__ mom_off,
                                                    const int64_t *__restrict__ tab_off, const float *__restrict__ tab,
                                                    const double *__restrict__ mom, KConst kc, int32_t nfreq, int32_t want_grad,
                                                    double *__restrict__ out, int64_t out_stride, int32_t *err) {
    const int e = blockIdx.y;
    const CellsDev *cl = cells + cfg_of[e];
    const int ncell = cl->ncell;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int4 rows = __ldg(reinterpret_cast<const int4 *>(cl->cellrows) + c);
    const float *tb = tab + tab_off[e] * NROW;
    const float *rFd = tb + (int64_t)rows.x * NROW, *rG = tb + (int64_t)rows.y * NROW, *rdG = tb + (int64_t)rows.z * NROW,
                *rFs = tb + (int64_t)rows.w * NROW;
    // the two non-trivial columns of A (the table values are the fp32 ones the per-pixel path uses); zero beyond nfreq
    double a1[CC_MAXF], a2[CC_MAXF];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 fd = __ldg(reinterpret_cast<const float4 *>(rFd) + q), g = __ldg(reinterpret_cast<const float4 *>(rG) + q),
                     fs = __ldg(reinterpret_cast<const float4 *>(rFs) + q);
        const float vfd[4] = {fd.x, fd.y, fd.z, fd.w}, vg[4] = {g.x, g.y, g.z, g.w}, vfs[4] = {fs.x, fs.y, fs.z, fs.w};
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const int f = 4 * q + h;
            if (f < CC_MAXF) {
                a1[f] = (f < nfreq) ? (double)vfd[h] * (double)vg[h] : 0.0;
                a2[f] = (f < nfreq) ? (double)vfs[h] : 0.0;
            }
        }
    }
    // u_i = T a_i (a_0 = 1) from the 120 unique moments
    const double *T = mom + mom_off[e] + c;
    double u0[CC_MAXF], u1[CC_MAXF], u2[CC_MAXF];
#pragma unroll
    for (int f = 0; f < CC_MAXF; ++f) {
        const double t = __ldg(T + (int64_t)cc_idx(f, f) * ncell);
        u0[f] = t; u1[f] = t * a1[f]; u2[f] = t * a2[f];
    }
#pragma unroll
    for (int f = 0; f < CC_MAXF; ++f) {
#pragma unroll
        for (int g = f + 1; g < CC_MAXF; ++g) {
            const double t = __ldg(T + (int64_t)cc_idx(f, g) * ncell);
            u0[f] += t; u0[g] += t;
            u1[f] = fma(t, a1[g], u1[f]); u1[g] = fma(t, a1[f], u1[g]);
            u2[f] = fma(t, a2[g], u2[f]); u2[g] = fma(t, a2[f], u2[g]);
        }
    }
    // B = A^T T A and V_th = U^T a'_th
    double b00 = 0, b01 = 0, b02 = 0, b11 = 0, b12 = 0, b22 = 0;
    double v1[3] = {0, 0, 0}, v2[3] = {0, 0, 0}, v3[3] = {0, 0, 0};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 dg4 = __ldg(reinterpret_cast<const float4 *>(rdG) + q);
        const float vdg[4] = {dg4.x, dg4.y, dg4.z, dg4.w};
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const int f = 4 * q + h;
            if (f < CC_MAXF) {
                const double x1 = a1[f], x2 = a2[f];
                b00 += u0[f]; b01 += u1[f]; b02 += u2[f];
                b11 = fma(x1, u1[f], b11); b12 = fma(x1, u2[f], b12); b22 = fma(x2, u2[f], b22);
                const double d1 = (double)kc.lnd[f] * x1, d2 = (double)vdg[h] * x1, d3 = (double)kc.lns[f] * x2;
                v1[0] = fma(d1, u0[f], v1[0]); v1[1] = fma(d1, u1[f], v1[1]); v1[2] = fma(d1, u2[f], v1[2]);
                v2[0] = fma(d2, u0[f], v2[0]); v2[1] = fma(d2, u1[f], v2[1]); v2[2] = fma(d2, u2[f], v2[2]);
                v3[0] = fma(d3, u0[f], v3[0]); v3[1] = fma(d3, u1[f], v3[1]); v3[2] = fma(d3, u2[f], v3[2]);
            }
        }
    }
    // M = A^T N^-1 A and P_th = A^T N^-1 a'_th from the columns
    double m00 = 0, m01 = 0, m02 = 0, m11 = 0, m12 = 0, m22 = 0;
    double p1[3] = {0, 0, 0}, p2[3] = {0, 0, 0}, p3[3] = {0, 0, 0};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float4 dg4 = __ldg(reinterpret_cast<const float4 *>(rdG) + q);
        const float vdg[4] = {dg4.x, dg4.y, dg4.z, dg4.w};
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const int f = 4 * q + h;
            if (f < CC_MAXF) {
                const double x1 = a1[f], x2 = a2[f];
                const double wf = (double)kc.w[f], wd = wf * x1, ws = wf * x2;
                m00 += wf; m01 += wd; m02 += ws; m11 += wd * x1; m12 += wd * x2; m22 += ws * x2;
                const double q1 = (double)kc.lnd[f] * wd, q2 = (double)vdg[h] * wd, q3 = (double)kc.lns[f] * ws;
                p1[0] += q1; p1[1] += q1 * x1; p1[2] += q1 * x2;
                p2[0] += q2; p2[1] += q2 * x1; p2[2] += q2 * x2;
                p3[0] += q3; p3[1] += q3 * x1; p3[2] += q3 * x2;
            }
        }
    }
    // M^-1 by cofactors (3 x 3 symmetric positive definite; cond ~ 5, R11)
    const double c00 = m11 * m22 - m12 * m12, c01 = m02 * m12 - m01 * m22, c02 = m01 * m12 - m02 * m11;
    const double c11 = m00 * m22 - m02 * m02, c12 = m01 * m02 - m00 * m12, c22 = m00 * m11 - m01 * m01;
    const double det = m00 * c00 + m01 * c01 + m02 * c02;
    const bool bad = !(det > 1e-12 * m00 * m11 * m22);
    if (bad) atomicOr(err, ERR_SINGULAR);
    const double id = 1.0 / det;
    const double i00 = c00 * id, i01 = c01 * id, i02 = c02 * id, i11 = c11 * id, i12 = c12 * id, i22 = c22 * id;
    // tr(M^-1 B)
    const double tr = i00 * b00 + i11 * b11 + i22 * b22 + 2.0 * (i01 * b01 + i02 * b02 + i12 * b12);
    double *o = out + (int64_t)e * out_stride + c;
    const int64_t cs_ = out_stride / 4;
    o[0] = bad ? CUDART_INF : -0.5 * tr;
    if (want_grad) {
        // X = M^-1 B M^-1: rows 1 (dust) and 2 (synchrotron) are all the gradient needs
        const double y10 = i01 * b00 + i11 * b01 + i12 * b02, y11 = i01 * b01 + i11 * b11 + i12 * b12, y12 = i01 * b02 + i11 * b12 + i12 * b22;
        const double y20 = i02 * b00 + i12 * b01 + i22 * b02, y21 = i02 * b01 + i12 * b11 + i22 * b12, y22 = i02 * b02 + i12 * b12 + i22 * b22;
        const double x10 = y10 * i00 + y11 * i01 + y12 * i02, x11 = y10 * i01 + y11 * i11 + y12 * i12, x12 = y10 * i02 + y11 * i12 + y12 * i22;
        const double x20 = y20 * i00 + y21 * i01 + y22 * i02, x21 = y20 * i01 + y21 * i11 + y22 * i12, x22 = y20 * i02 + y21 * i12 + y22 * i22;
        o[cs_] = (x10 * p1[0] + x11 * p1[1] + x12 * p1[2]) - (i01 * v1[0] + i11 * v1[1] + i12 * v1[2]);
        o[2 * cs_] = (x10 * p2[0] + x11 * p2[1] + x12 * p2[2]) - (i01 * v2[0] + i11 * v2[1] + i12 * v2[2]);
        o[3 * cs_] = (x20 * p3[0] + x21 * p3[1] + x22 * p3[2]) - (i02 * v3[0] + i12 * v3[1] + i22 * v3[2]);
    }
}

// Ordered sums of the per-cell terms onto clusters (grad) and regions (nll).  A cluster with at most CC_LONG cells: one
// thread, cells in ascending order.  Longer lists (every region; the clusters of maps with a handful of patches) are
// summed by a whole block: thread i adds the cells i, i+128, ... of the list in ascending order, the 32 lane sums of a
// warp are combined by a fixed xor-shuffle tree and the four warp sums left to right.  Which way a cluster goes depends
// on its cell count only: deterministic and independent of the batch.
// grid = (ceil(ktot_max / 128) [cluster blocks, want_grad only] + nregion [region blocks], batch), block = 128.
constexpr int CC_LONG = 64;
__device__ __forceinline__ double cc_block_sum(const double *__restrict__ src, const int32_t *__restrict__ list, int a, int b, double *wsum) {
    double acc = 0.0;
#pragma unroll 8
    for (int q = a + (int)threadIdx.x; q < b; q += 128) acc += src[__ldg(list + q)];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __syncthreads();   // wsum is free again
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    __syncthreads();
    return ((wsum[0] + wsum[1]) + wsum[2]) + wsum[3];
}
__global__ void __launch_bounds__(128) k_cc_reduce(const CfgDev *__restrict__ cfgs, const CellsDev *__restrict__ cells,
                                                   const int32_t *__restrict__ cfg_of, const int64_t *__restrict__ param_off,
                                                   const double *__restrict__ out, int64_t out_stride, int32_t nregion,
                                                   int32_t want_grad, double *__restrict__ nll, double *__restrict__ grad) {
    __shared__ double wsum[4];
    __shared__ int32_t s_long[128][3];   // (first, end, term) of this block's long clusters, by thread
    __shared__ int32_t s_who[128], s_nlong;
    const int e = blockIdx.y;
    const CfgDev *cf = cfgs + cfg_of[e];
    const CellsDev *cl = cells + cfg_of[e];
    const double *o = out + (int64_t)e * out_stride;
    const int64_t cs_ = out_stride / 4;
    const int nblk_cluster = (int)gridDim.x - nregion;
    if ((int)blockIdx.x < nblk_cluster) {
        const int ktot = cf->ktot;
        if ((int)(blockIdx.x * blockDim.x) >= ktot) return;   // block-uniform
        if (threadIdx.x == 0) s_nlong = 0;
        __syncthreads();
        const int v = blockIdx.x * blockDim.x + threadIdx.x;
        const int64_t dst0 = param_off[e] + (int64_t)blockIdx.x * blockDim.x;
        if (v < ktot) {
            int t, k;
            if (v < cf->K[0]) { t = 0; k = v; }
            else if (v < cf->K[0] + cf->K[1]) { t = 1; k = v - cf->K[0]; }
            else { t = 2; k = v - cf->K[0] - cf->K[1]; }
            const int a = __ldg(cl->kptr[t] + k), b = __ldg(cl->kptr[t] + k + 1);
            if (b - a <= CC_LONG) {
                const double *src = o + (int64_t)(t + 1) * cs_;
                const int32_t *list = cl->klist[t];
                double acc = 0.0;
#pragma unroll 8
                for (int q = a; q < b; ++q) acc += src[__ldg(list + q)];
                grad[dst0 + threadIdx.x] = acc;
            } else {
                s_long[threadIdx.x][0] = a; s_long[threadIdx.x][1] = b; s_long[threadIdx.x][2] = t;
                s_who[atomicAdd(&s_nlong, 1)] = threadIdx.x;
            }
        }
        __syncthreads();
        const int nlong = s_nlong;
        for (int i = 0; i < nlong; ++i) {   // in any order: every sum is on its own
            const int who = s_who[i], t = s_long[who][2];
            const double tot = cc_block_sum(o + (int64_t)(t + 1) * cs_, cl->klist[t], s_long[who][0], s_long[who][1], wsum);
            if (threadIdx.x == 0) grad[dst0 + who] = tot;
        }
    } else {
        const int r = (int)blockIdx.x - nblk_cluster;
        const int a = __ldg(cl->kptr[3] + r), b = __ldg(cl->kptr[3] + r + 1);
        const double tot = cc_block_sum(o, cl->klist[3], a, b, wsum);
        if (threadIdx.x == 0) nll[(int64_t)e * nregion + r] = tot;
    }
}

}  // namespace cs
