// cs_math.cuh -- the arithmetic of the fused kernels, written once.
//
// A consumer thread evaluates the two positions (2t, 2t+1) of its tile at once: every per-pixel quantity is a float2
// whose lanes are the two pixels, and every operation on it is one packed FFMA2 / FMUL2 / FADD2 (sm_100).  Band sums
// run sequentially over the bands f = 0 .. nfreq-1 inside each lane.
//   sorted-cell kernel  the two pixels share their cell: the per-cell part below is evaluated once per cell by a builder
//                       lane in scalar arithmetic (T = float) and enters the per-pixel part as scalars that the packed
//                       instructions broadcast to both lanes;
//   direct kernel       every pixel is its own cell: the per-cell part runs packed too (T = float2, lanes = pixels).
// Both call exactly these functions, and a packed instruction rounds each lane like the scalar one, so a pixel-eval
// gives the same bits in either kernel.  That is what makes results independent of the kernel form.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"

namespace cs {

__device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float2 mul_(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add_(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fma_(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
// scalar operand of a packed instruction: (x, x); ptxas folds it into the instruction's broadcast operand form
__device__ __forceinline__ float2 mul_(float a, float2 b) { return __fmul2_rn(make_float2(a, a), b); }
__device__ __forceinline__ float2 fma_(float a, float2 b, float2 c) { return __ffma2_rn(make_float2(a, a), b, c); }
__device__ __forceinline__ float2 fma_(float2 a, float b, float2 c) { return __ffma2_rn(a, make_float2(b, b), c); }
__device__ __forceinline__ float neg_(float a) { return -a; }
__device__ __forceinline__ float2 neg_(float2 a) { return make_float2(-a.x, -a.y); }
template <class T> __device__ __forceinline__ T zero_();
template <> __device__ __forceinline__ float zero_<float>() { return 0.f; }
template <> __device__ __forceinline__ float2 zero_<float2>() { return make_float2(0.f, 0.f); }

// 1/x for x > 0 in normal range: MUFU.RCP plus one Newton step (error below 1 ulp; no slow-path branch).
__device__ __forceinline__ float fast_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return __fmaf_rn(r, __fmaf_rn(-x, r, 1.0f), r);
}
__device__ __forceinline__ float2 fast_rcp(float2 x) { return make_float2(fast_rcp(x.x), fast_rcp(x.y)); }
__device__ __forceinline__ float flag_bad(float d1, float M11, float d2, float M22) {
    return ((d1 > PIVOT_RTOL * M11) && (d2 > PIVOT_RTOL * M22)) ? 0.f : 1.f;
}
__device__ __forceinline__ float2 flag_bad(float2 d1, float2 M11, float2 d2, float2 M22) {
    return make_float2(flag_bad(d1.x, M11.x, d2.x, M22.x), flag_bad(d1.y, M11.y, d2.y, M22.y));
}

// ---- per cell (cluster triple): Eq. 2 columns -> weighted columns, M = A^T N^-1 A (L233), its LDL^T, P ------------
template <class T>
struct CellSums {   // running band sums; m00 = sum_f w_f is a constant of the data set
    T m01, m02, m11, m12, m22;
    T p10, p11, p12, p20, p21, p22, p30, p31, p32;
};
template <class T>
__device__ __forceinline__ void cell_sums_zero(CellSums<T> &S) {
    const T z = zero_<T>();
    S.m01 = S.m02 = S.m11 = S.m12 = S.m22 = z;
    S.p10 = S.p11 = S.p12 = S.p20 = S.p21 = S.p22 = S.p30 = S.p31 = S.p32 = z;
}
template <class T>
struct CellCols {   // the weighted columns of one band: w a_d, w da_d/dbeta_d, w da_d/dT_d, w a_s, w da_s/dbeta_s
    T wd, u1, u2, ws, u3;
};
// One band of a cell: a_d = Fd' G (Eq. 2), a_s = Fs'; accumulates M and (GRAD) P_{theta,c} = sum_f w_f (da_f/dtheta) A_{f,c}.
template <bool GRAD, class T>
__device__ __forceinline__ void cell_band(CellSums<T> &S, CellCols<T> &C, T Fd, T G, T dG, T as, float w, float lnd, float lns) {
    const T ad = mul_(Fd, G);
    C.wd = mul_(w, ad);
    C.ws = mul_(w, as);
    S.m01 = add_(S.m01, C.wd); S.m02 = add_(S.m02, C.ws);
    S.m11 = fma_(C.wd, ad, S.m11); S.m12 = fma_(C.wd, as, S.m12); S.m22 = fma_(C.ws, as, S.m22);
    if (GRAD) {
        C.u1 = mul_(lnd, C.wd);
        C.u2 = mul_(dG, C.wd);
        C.u3 = mul_(lns, C.ws);
        S.p10 = add_(S.p10, C.u1); S.p11 = fma_(C.u1, ad, S.p11); S.p12 = fma_(C.u1, as, S.p12);
        S.p20 = add_(S.p20, C.u2); S.p21 = fma_(C.u2, ad, S.p21); S.p22 = fma_(C.u2, as, S.p22);
        S.p30 = add_(S.p30, C.u3); S.p31 = fma_(C.u3, ad, S.p31); S.p32 = fma_(C.u3, as, S.p32);
    } else {
        C.u1 = C.u2 = C.u3 = zero_<T>();
    }
}
template <class T>
struct CellScal {   // what a pixel-eval needs from its cell besides the columns
    T l10, l20, l21, id1, id2;
    T P10, P11, P12, P20, P21, P22, P30, P31, P32;
    T bad;          // 1 when a pivot of M is not above PIVOT_RTOL of its diagonal entry (CS_ESINGULAR), else 0
};
template <bool GRAD, class T>
__device__ __forceinline__ void cell_finish(const CellSums<T> &S, float inv_m00, CellScal<T> &C) {
    C.l10 = mul_(inv_m00, S.m01); C.l20 = mul_(inv_m00, S.m02);
    const T d1 = fma_(neg_(C.l10), S.m01, S.m11);
    const T t12 = fma_(neg_(C.l10), S.m02, S.m12);
    C.id1 = fast_rcp(d1);
    C.l21 = mul_(t12, C.id1);
    const T d2 = fma_(neg_(C.l21), t12, fma_(neg_(C.l20), S.m02, S.m22));
    C.id2 = fast_rcp(d2);
    C.bad = flag_bad(d1, S.m11, d2, S.m22);
    const T z = zero_<T>();
    C.P10 = C.P11 = C.P12 = C.P20 = C.P21 = C.P22 = C.P30 = C.P31 = C.P32 = z;
    if (GRAD) {
        C.P10 = S.p10; C.P11 = S.p11; C.P12 = S.p12;
        C.P20 = S.p20; C.P21 = S.p21; C.P22 = S.p22;
        C.P30 = S.p30; C.P31 = S.p31; C.P32 = S.p32;
    }
}

// ---- per pixel pair: b = A^T N^-1 d (Eq. 5), c = (dA/dtheta)^T N^-1 d, solve, likelihood and gradient terms --------
struct PixSums {   // lanes = the thread's two pixels
    float2 bq0, bq1, bq2, bu0, bu1, bu2;
    float2 cq1, cq2, cq3, cu1, cu2, cu3;
};
__device__ __forceinline__ void pix_sums_zero(PixSums &A) {
    const float2 z = make_float2(0.f, 0.f);
    A.bq0 = A.bq1 = A.bq2 = A.bu0 = A.bu1 = A.bu2 = z;
    A.cq1 = A.cq2 = A.cq3 = A.cu1 = A.cu2 = A.cu3 = z;
}
// One band: the weighted columns of the pixels' cell(s) (T = float: one cell for both; float2: one per pixel) against
// the pixels' Q and U data.
template <bool GRAD, class T>
__device__ __forceinline__ void pix_band(PixSums &A, const CellCols<T> &C, float w, float2 dq, float2 du) {
    A.bq0 = fma_(w, dq, A.bq0); A.bq1 = fma_(C.wd, dq, A.bq1); A.bq2 = fma_(C.ws, dq, A.bq2);
    A.bu0 = fma_(w, du, A.bu0); A.bu1 = fma_(C.wd, du, A.bu1); A.bu2 = fma_(C.ws, du, A.bu2);
    if (GRAD) {
        A.cq1 = fma_(C.u1, dq, A.cq1); A.cq2 = fma_(C.u2, dq, A.cq2); A.cq3 = fma_(C.u3, dq, A.cq3);
        A.cu1 = fma_(C.u1, du, A.cu1); A.cu2 = fma_(C.u2, du, A.cu2); A.cu3 = fma_(C.u3, du, A.cu3);
    }
}
__device__ __forceinline__ float2 sel_inf(float bad, float2 v) { return bad != 0.f ? make_float2(CUDART_INF_F, CUDART_INF_F) : v; }
__device__ __forceinline__ float2 sel_inf(float2 bad, float2 v) {
    return make_float2(bad.x != 0.f ? CUDART_INF_F : v.x, bad.y != 0.f ? CUDART_INF_F : v.y);
}
// LDL^T solve for one Stokes parameter; returns b . s
template <class T>
__device__ __forceinline__ float2 solve1(float2 b0, float2 b1, float2 b2, const CellScal<T> &C, float inv_m00, float2 (&s)[3]) {
    const float2 y1 = fma_(neg_(C.l10), b0, b1);
    const float2 y2 = fma_(neg_(C.l21), y1, fma_(neg_(C.l20), b0, b2));
    const float2 z0 = mul_(inv_m00, b0), z1 = mul_(C.id1, y1), z2 = mul_(C.id2, y2);
    s[2] = z2;
    s[1] = fma_(neg_(C.l21), z2, z1);
    s[0] = fma_(neg_(C.l20), s[2], fma_(neg_(C.l10), s[1], z0));
    return fma_(b0, z0, fma_(y1, z1, mul_(y2, z2)));
}
// LDL^T solves for Q and U, ll = -1/2 sum_S b_S . s_S (Eq. 6); +inf when the cell's M is flagged.
template <class T>
__device__ __forceinline__ void pix_solve(const PixSums &A, const CellScal<T> &C, float inv_m00, float2 (&sq)[3], float2 (&su)[3], float2 &ll) {
    const float2 lq = solve1(A.bq0, A.bq1, A.bq2, C, inv_m00, sq);
    const float2 lu = solve1(A.bu0, A.bu1, A.bu2, C, inv_m00, su);
    ll = sel_inf(C.bad, mul_(-0.5f, add_(lq, lu)));
}
// g_theta = - sum_S s_{S,c} ( c_{S,theta} - P_theta . s_S )   (Eq. 17 with r = d - A s expanded, s held fixed)
template <class T>
__device__ __forceinline__ void pix_grad_terms(const PixSums &A, const CellScal<T> &C, const float2 (&sq)[3], const float2 (&su)[3],
                                               float2 &g_bd, float2 &g_td, float2 &g_bs) {
    const float2 eq1 = fma_(neg_(C.P12), sq[2], fma_(neg_(C.P11), sq[1], fma_(neg_(C.P10), sq[0], A.cq1)));
    const float2 eu1 = fma_(neg_(C.P12), su[2], fma_(neg_(C.P11), su[1], fma_(neg_(C.P10), su[0], A.cu1)));
    const float2 eq2 = fma_(neg_(C.P22), sq[2], fma_(neg_(C.P21), sq[1], fma_(neg_(C.P20), sq[0], A.cq2)));
    const float2 eu2 = fma_(neg_(C.P22), su[2], fma_(neg_(C.P21), su[1], fma_(neg_(C.P20), su[0], A.cu2)));
    const float2 eq3 = fma_(neg_(C.P32), sq[2], fma_(neg_(C.P31), sq[1], fma_(neg_(C.P30), sq[0], A.cq3)));
    const float2 eu3 = fma_(neg_(C.P32), su[2], fma_(neg_(C.P31), su[1], fma_(neg_(C.P30), su[0], A.cu3)));
    g_bd = neg_(fma_(sq[1], eq1, mul_(su[1], eu1)));
    g_td = neg_(fma_(sq[1], eq2, mul_(su[1], eu2)));
    g_bs = neg_(fma_(sq[2], eq3, mul_(su[2], eu3)));
}

// chi^2 of the pixels' GLS residual, a second pass over the bands once s is known: r_S = d_S - A s_S,
// chi2 = sum_S sum_f w_f r_{S,f}^2 = 2 nll + d^T N^-1 d.  Unlike -1/2 b.s (a difference of large numbers once the
// parameter-independent d^T N^-1 d is taken out) it resolves small changes of the objective: the line search runs on it.
// The columns are recovered from the weighted ones: a_d = (w a_d) / w, a_s = (w a_s) / w.
template <class T>
__device__ __forceinline__ void pix_chi2_band(float2 &xq, float2 &xu, const float2 (&sq)[3], const float2 (&su)[3], T wd, T ws,
                                              float w, float invw, float2 dq, float2 du) {
    const T ad = mul_(invw, wd), as = mul_(invw, ws);
    const float2 rq = fma_(neg_(sq[2]), as, fma_(neg_(sq[1]), ad, add_(dq, neg_(sq[0]))));
    const float2 ru = fma_(neg_(su[2]), as, fma_(neg_(su[1]), ad, add_(du, neg_(su[0]))));
    xq = fma_(mul_(w, rq), rq, xq);
    xu = fma_(mul_(w, ru), ru, xu);
}

// ---- ordered fp64 sums of the rank-ordered term rows (a3, first level) --------------------------------------------
// A chunk is <= CHUNK_LEN consecutive ranks of one cluster, missing ranks counting as zero, combined as the tree
// ((x0+x1)+(x2+x3)) + ((x4+x5)+(x6+x7)) in fp64.  In the sorted layout ranks 2i and 2i+1 always belong to one
// thread, which adds them itself: the reducer then sees the four pair sums y_i and forms (y0+y1)+(y2+y3).
__device__ __forceinline__ double pair_sum(float a, float b) { return (double)a + (double)b; }
__device__ __forceinline__ double chunk_tree(double y0, double y1, double y2, double y3) { return (y0 + y1) + (y2 + y3); }
__device__ __forceinline__ double chunk_sum(const float *term, int start, int len) {
    float x[CHUNK_LEN];
#pragma unroll
    for (int k = 0; k < CHUNK_LEN; ++k) x[k] = (k < len) ? term[start + k] : 0.f;
    return chunk_tree(pair_sum(x[0], x[1]), pair_sum(x[2], x[3]), pair_sum(x[4], x[5]), pair_sum(x[6], x[7]));
}
// Sum of a segment (<= SEG_MAX ranks of one cluster): its chunk sums, left to right.
__device__ __forceinline__ double segment_sum(const float *term, int start, int len) {
    double acc = chunk_sum(term, start, min(len, CHUNK_LEN));
    for (int o = CHUNK_LEN; o < len; o += CHUNK_LEN) acc += chunk_sum(term, start + o, min(len - o, CHUNK_LEN));
    return acc;
}

}  // namespace cs
