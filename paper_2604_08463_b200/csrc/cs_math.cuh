// cs_math.cuh -- the per-pixel arithmetic of the fused kernels, written once.
//
// Both forms of the fused kernel (k_like_cell: per-cell part by builder threads, per-pixel part by consumer threads;
// k_like: both parts by the pixel's own thread) call exactly these functions in exactly this order, so a pixel's
// likelihood and gradient terms are bit-identical whichever form evaluates it.  That is what makes the result
// independent of how entries are grouped into batches although the library picks the kernel form per group.
//
// All packed operations (FFMA2 / FMUL2 / FADD2 on sm_100) carry two consecutive bands (2j, 2j+1); band 15 is a zero pad.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"

namespace cs {

__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 dup2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float hsum(float2 a) { return a.x + a.y; }

// 1/x for x > 0 in normal range: MUFU.RCP plus one Newton step (error below 1 ulp; no slow-path branch).
__device__ __forceinline__ float fast_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}

// ---- per cell (cluster triple): Eq. 2 columns -> weighted column, M = A^T N^-1 A (L233), its LDL^T, P -------------
struct CellSums {   // band-pair partial sums; m00 = sum_f w_f is a constant of the data set
    float2 m01, m02, m11, m12, m22;
    float2 p10, p11, p12, p20, p21, p22, p30, p31, p32;
};
__device__ __forceinline__ void cell_sums_zero(CellSums &S) {
    const float2 z = make_float2(0.f, 0.f);
    S.m01 = S.m02 = S.m11 = S.m12 = S.m22 = z;
    S.p10 = S.p11 = S.p12 = S.p20 = S.p21 = S.p22 = S.p30 = S.p31 = S.p32 = z;
}
// One band pair j of a cell: a_d = Fd' G (Eq. 2), wd = w a_d, ws = w a_s; accumulates M and (GRAD) P.  Returns wd.
template <bool GRAD>
__device__ __forceinline__ float2 cell_pair(CellSums &S, float2 Fd, float2 G, float2 dG, float2 as, float2 w, float2 lnd, float2 lns) {
    const float2 ad = mul2(Fd, G);
    const float2 wd = mul2(w, ad);
    const float2 ws = mul2(w, as);
    S.m01 = add2(S.m01, wd); S.m02 = add2(S.m02, ws);
    S.m11 = fma2(wd, ad, S.m11); S.m12 = fma2(wd, as, S.m12); S.m22 = fma2(ws, as, S.m22);
    if (GRAD) {
        const float2 u1 = mul2(lnd, wd);      // w da_d/dbeta_d
        const float2 u2 = mul2(dG, wd);       // w da_d/dT_d
        const float2 u3 = mul2(lns, ws);      // w da_s/dbeta_s
        S.p10 = add2(S.p10, u1); S.p11 = fma2(u1, ad, S.p11); S.p12 = fma2(u1, as, S.p12);
        S.p20 = add2(S.p20, u2); S.p21 = fma2(u2, ad, S.p21); S.p22 = fma2(u2, as, S.p22);
        S.p30 = add2(S.p30, u3); S.p31 = fma2(u3, ad, S.p31); S.p32 = fma2(u3, as, S.p32);
    }
    return wd;
}
struct CellScal {   // what a pixel-eval needs from its cell besides the columns
    float l10, l20, l21, id1, id2;
    float P10, P11, P12, P20, P21, P22, P30, P31, P32;
    float bad;      // 1 when a pivot of M is not above PIVOT_RTOL of its diagonal entry (CS_ESINGULAR), else 0
};
template <bool GRAD>
__device__ __forceinline__ void cell_finish(const CellSums &S, float inv_m00, CellScal &C) {
    const float M01 = hsum(S.m01), M02 = hsum(S.m02), M11 = hsum(S.m11), M12 = hsum(S.m12), M22 = hsum(S.m22);
    C.l10 = M01 * inv_m00; C.l20 = M02 * inv_m00;
    const float d1 = fmaf(-C.l10, M01, M11);
    const float t12 = fmaf(-C.l10, M02, M12);
    C.id1 = fast_rcp(d1);
    C.l21 = t12 * C.id1;
    const float d2 = fmaf(-C.l21, t12, fmaf(-C.l20, M02, M22));
    C.id2 = fast_rcp(d2);
    C.bad = ((d1 > PIVOT_RTOL * M11) && (d2 > PIVOT_RTOL * M22)) ? 0.f : 1.f;
    C.P10 = C.P11 = C.P12 = C.P20 = C.P21 = C.P22 = C.P30 = C.P31 = C.P32 = 0.f;
    if (GRAD) {
        C.P10 = hsum(S.p10); C.P11 = hsum(S.p11); C.P12 = hsum(S.p12);
        C.P20 = hsum(S.p20); C.P21 = hsum(S.p21); C.P22 = hsum(S.p22);
        C.P30 = hsum(S.p30); C.P31 = hsum(S.p31); C.P32 = hsum(S.p32);
    }
}

// ---- per pixel: b = A^T N^-1 d (Eq. 5), c = (dA/dtheta)^T N^-1 d, solve, likelihood and gradient terms ------------
struct PixSums {
    float2 bq0, bq1, bq2, bu0, bu1, bu2;
    float2 cq1, cq2, cq3, cu1, cu2, cu3;
};
__device__ __forceinline__ void pix_sums_zero(PixSums &A) {
    const float2 z = make_float2(0.f, 0.f);
    A.bq0 = A.bq1 = A.bq2 = A.bu0 = A.bu1 = A.bu2 = z;
    A.cq1 = A.cq2 = A.cq3 = A.cu1 = A.cu2 = A.cu3 = z;
}
// One band pair: wd = w a_d of the pixel's cell, fs = Fs'[k2] = a_s, dg = dlnG[k1]; dq, du = the pixel's Q and U data.
template <bool GRAD>
__device__ __forceinline__ void pix_pair(PixSums &A, float2 wd, float2 fs, float2 dg, float2 w, float2 lnd, float2 lns, float2 dq, float2 du) {
    const float2 ws = mul2(w, fs);
    A.bq0 = fma2(w, dq, A.bq0); A.bq1 = fma2(wd, dq, A.bq1); A.bq2 = fma2(ws, dq, A.bq2);
    A.bu0 = fma2(w, du, A.bu0); A.bu1 = fma2(wd, du, A.bu1); A.bu2 = fma2(ws, du, A.bu2);
    if (GRAD) {
        const float2 u2 = mul2(dg, wd);
        const float2 u1 = mul2(lnd, wd), u3 = mul2(lns, ws);
        A.cq1 = fma2(u1, dq, A.cq1); A.cq2 = fma2(u2, dq, A.cq2); A.cq3 = fma2(u3, dq, A.cq3);
        A.cu1 = fma2(u1, du, A.cu1); A.cu2 = fma2(u2, du, A.cu2); A.cu3 = fma2(u3, du, A.cu3);
    }
}
// LDL^T solves for Q and U, ll = -1/2 sum_S b_S . s_S (Eq. 6); +inf when the cell's M is flagged.
__device__ __forceinline__ void pix_solve(const PixSums &A, const CellScal &C, float inv_m00, float (&sq)[3], float (&su)[3], float &ll) {
    {
        const float b0 = hsum(A.bq0), b1 = hsum(A.bq1), b2 = hsum(A.bq2);
        const float y1 = fmaf(-C.l10, b0, b1);
        const float y2 = fmaf(-C.l21, y1, fmaf(-C.l20, b0, b2));
        const float z0 = b0 * inv_m00, z1 = y1 * C.id1, z2 = y2 * C.id2;
        sq[2] = z2; sq[1] = fmaf(-C.l21, z2, z1); sq[0] = fmaf(-C.l20, sq[2], fmaf(-C.l10, sq[1], z0));
        ll = fmaf(b0, z0, fmaf(y1, z1, y2 * z2));
    }
    {
        const float b0 = hsum(A.bu0), b1 = hsum(A.bu1), b2 = hsum(A.bu2);
        const float y1 = fmaf(-C.l10, b0, b1);
        const float y2 = fmaf(-C.l21, y1, fmaf(-C.l20, b0, b2));
        const float z0 = b0 * inv_m00, z1 = y1 * C.id1, z2 = y2 * C.id2;
        su[2] = z2; su[1] = fmaf(-C.l21, z2, z1); su[0] = fmaf(-C.l20, su[2], fmaf(-C.l10, su[1], z0));
        ll += fmaf(b0, z0, fmaf(y1, z1, y2 * z2));
    }
    ll *= -0.5f;
    if (C.bad != 0.f) ll = CUDART_INF_F;
}
// g_theta = - sum_S s_{S,c} ( c_{S,theta} - P_theta . s_S )   (Eq. 17 with r = d - A s expanded, s held fixed)
__device__ __forceinline__ void pix_grad_terms(const PixSums &A, const CellScal &C, const float (&sq)[3], const float (&su)[3],
                                               float &g_bd, float &g_td, float &g_bs) {
    const float eq1 = fmaf(-C.P12, sq[2], fmaf(-C.P11, sq[1], fmaf(-C.P10, sq[0], hsum(A.cq1))));
    const float eu1 = fmaf(-C.P12, su[2], fmaf(-C.P11, su[1], fmaf(-C.P10, su[0], hsum(A.cu1))));
    const float eq2 = fmaf(-C.P22, sq[2], fmaf(-C.P21, sq[1], fmaf(-C.P20, sq[0], hsum(A.cq2))));
    const float eu2 = fmaf(-C.P22, su[2], fmaf(-C.P21, su[1], fmaf(-C.P20, su[0], hsum(A.cu2))));
    const float eq3 = fmaf(-C.P32, sq[2], fmaf(-C.P31, sq[1], fmaf(-C.P30, sq[0], hsum(A.cq3))));
    const float eu3 = fmaf(-C.P32, su[2], fmaf(-C.P31, su[1], fmaf(-C.P30, su[0], hsum(A.cu3))));
    g_bd = -fmaf(sq[1], eq1, su[1] * eu1);
    g_td = -fmaf(sq[1], eq2, su[1] * eu2);
    g_bs = -fmaf(sq[2], eq3, su[2] * eu3);
}

// chi^2 of the pixel's GLS residual, a second pass over the bands once s is known: r_S = d_S - A s_S,
// chi2 = sum_S sum_f w_f r_{S,f}^2 = 2 nll + d^T N^-1 d.  Unlike -1/2 b.s (a difference of large numbers once the
// parameter-independent d^T N^-1 d is taken out) it resolves small changes of the objective: the line search runs on it.
struct ChiSums {
    float2 q, u;
};
struct ChiCoef {   // -s_{S,c} duplicated into both lanes
    float2 q0, q1, q2, u0, u1, u2;
};
__device__ __forceinline__ void chi_coef(const float (&sq)[3], const float (&su)[3], ChiCoef &K) {
    K.q0 = dup2(-sq[0]); K.q1 = dup2(-sq[1]); K.q2 = dup2(-sq[2]);
    K.u0 = dup2(-su[0]); K.u1 = dup2(-su[1]); K.u2 = dup2(-su[2]);
}
// wd = w a_d of the pixel's cell (a_d is recovered as wd / w), fs = a_s
__device__ __forceinline__ void pix_chi2_pair(ChiSums &X, const ChiCoef &K, float2 wd, float2 fs, float2 w, float2 invw, float2 dq, float2 du) {
    const float2 ad = mul2(wd, invw);
    const float2 rq = fma2(K.q2, fs, fma2(K.q1, ad, add2(dq, K.q0)));
    const float2 ru = fma2(K.u2, fs, fma2(K.u1, ad, add2(du, K.u0)));
    X.q = fma2(mul2(w, rq), rq, X.q);
    X.u = fma2(mul2(w, ru), ru, X.u);
}

// ---- ordered fp64 sums of the rank-ordered term rows (a3, first level) --------------------------------------------
// Sum of a chunk of <= CHUNK_LEN consecutive ranks: elements are taken in an order rotated by the chunk's position
// (bank spreading for the reducer warps; a fixed function of the plan) and combined as (x0+x4)+(x1+x5) | (x2+x6)+(x3+x7).
__device__ __forceinline__ double chunk_sum(const float *term, int start, int len) {
    const int rot = (start >> 3) & (CHUNK_LEN - 1);
    float x[CHUNK_LEN];
#pragma unroll
    for (int k = 0; k < CHUNK_LEN; ++k) {
        const int j = (k + rot) & (CHUNK_LEN - 1);
        x[k] = (j < len) ? term[start + j] : 0.f;
    }
    const double a0 = (double)x[0] + (double)x[4], a1 = (double)x[1] + (double)x[5];
    const double a2 = (double)x[2] + (double)x[6], a3 = (double)x[3] + (double)x[7];
    return (a0 + a1) + (a2 + a3);
}
// Sum of a segment (<= SEG_MAX ranks of one cluster): its chunk sums, left to right.
__device__ __forceinline__ double segment_sum(const float *term, int start, int len) {
    double acc = chunk_sum(term, start, min(len, CHUNK_LEN));
    for (int o = CHUNK_LEN; o < len; o += CHUNK_LEN) acc += chunk_sum(term, start + o, min(len - o, CHUNK_LEN));
    return acc;
}

}  // namespace cs
