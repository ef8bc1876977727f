// cs_optim.cuh -- a5: device-resident fixed-budget AdaTopK (App. A, Alg. 1; readings R13/R14 of
// DESIGN.md).  Every batch entry is an independent bounded minimisation over its own parameter block.  All state
// lives on the device in fp64; the host only enqueues kernels (no synchronisation, no data-dependent launches).
//
// One iteration (Alg. 1):
//   y = (x - l)/(u - l), g_int = g * (u - l)                                   A1, L509-L513, Alg. 1 line 3
//   release the n = max(1, floor(topk n_bound)) bound parameters pushed hardest into the feasible region
//                                                                                A2-A3, L519-L537; topk = 0 (L249, L535): one
//   g_proj = g_int * (p == 0)                                                    line 8
//   if |g_proj| outside [safe_lo, safe_hi]: f = 1/|g_proj|; L,g_proj *= f; m *= f; v *= f^2     A4, L541-L546
//   AdaBelief direction (Zhuang et al. 2020), masked by p == 0                   lines 14-16
//   alpha_max = distance to the nearest bound along the direction                line 17
//   backtracking line search on alpha in (0, min(1, alpha_max)]                  line 18, L263
//   y += alpha d; pin the limiting parameter when alpha == alpha_max             lines 19-25
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cs {

struct OptWork {
    double *y = nullptr, *x = nullptr, *xt = nullptr, *dir = nullptr, *m = nullptr, *v = nullptr, *grad = nullptr;
    const double *lo = nullptr, *hi = nullptr;
    int8_t *pivot = nullptr;
    double *nll_reg = nullptr, *nll_reg_t = nullptr;
    double *Lcur = nullptr, *Lt_acc = nullptr;   // 1/2 chi^2 at the current point / at the accepted trial point
    double *L0 = nullptr, *gd = nullptr, *amax = nullptr, *alpha = nullptr, *alpha_acc = nullptr, *cscale = nullptr;
    long long *ilim = nullptr;
    int32_t *accepted = nullptr;
    int32_t *iter = nullptr;   // device-side iteration counter (the loop body is replayed as a CUDA graph)
    // L-BFGS back-end (f4(i)): unconstrained variable z, its gradient at the current point, the history ring
    double *z = nullptr, *gz = nullptr, *S = nullptr, *Y = nullptr;   // S, Y: [hist + 1][nparam] (ring; one slot is scratch)
    double *sy = nullptr;                                             // [hist + 1][batch] s.yv of each stored pair
    int32_t *hcount = nullptr, *hhead = nullptr, *moved = nullptr;    // [batch] pairs stored, next slot, last step accepted
    int32_t hist = 0;                                                 // history slots allocated
    int64_t lbfgs_bytes = 0;                                          // device bytes of the L-BFGS arrays above
};

struct OptShape {
    int64_t nparam;
    int32_t batch, nregion, ktot_max;
    const int64_t *param_off;
};

struct OptHyper {
    double lr, beta1, beta2, eps, c1, safe_lo, safe_hi, ls_noise, topk;
    int32_t ls_max;
};

inline void opt_free(OptWork &w) {
    cudaFree(w.y); cudaFree(w.x); cudaFree(w.xt); cudaFree(w.dir); cudaFree(w.m); cudaFree(w.v); cudaFree(w.grad);
    cudaFree(w.pivot); cudaFree(w.nll_reg); cudaFree(w.nll_reg_t); cudaFree(w.L0); cudaFree(w.gd); cudaFree(w.amax);
    cudaFree(w.alpha); cudaFree(w.alpha_acc); cudaFree(w.cscale); cudaFree(w.ilim); cudaFree(w.accepted); cudaFree(w.iter); cudaFree(w.Lcur); cudaFree(w.Lt_acc);
    cudaFree(w.z); cudaFree(w.gz); cudaFree(w.S); cudaFree(w.Y); cudaFree(w.sy); cudaFree(w.hcount); cudaFree(w.hhead); cudaFree(w.moved);
    w = OptWork();
}

// returns 0 ok, 1 out of memory
inline int opt_alloc(OptWork &w, int64_t nparam, int32_t batch, int32_t nregion, int64_t *bytes) {
    const size_t np = (size_t)(nparam > 0 ? nparam : 1) * sizeof(double), nb = (size_t)batch * sizeof(double);
    bool ok = true;
    ok &= cudaMalloc((void **)&w.y, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.x, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.xt, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.dir, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.m, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.v, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.grad, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.pivot, (size_t)(nparam > 0 ? nparam : 1)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.nll_reg, nb * nregion) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.nll_reg_t, nb * nregion) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.L0, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.gd, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.amax, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.alpha, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.alpha_acc, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.cscale, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.ilim, (size_t)batch * sizeof(long long)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.accepted, (size_t)batch * sizeof(int32_t)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.iter, sizeof(int32_t)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.Lcur, nb) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.Lt_acc, nb) == cudaSuccess;
    if (!ok) { opt_free(w); return 1; }
    *bytes = (int64_t)(7 * np + nparam + 2 * nb * nregion + 7 * nb + (size_t)batch * 4);
    return 0;
}

// workspace of the L-BFGS back-end, allocated on its first use (or when a longer history is asked for)
inline int opt_alloc_lbfgs(OptWork &w, int64_t nparam, int32_t batch, int32_t hist, int64_t *bytes) {
    if (w.z && w.hist >= hist) return 0;
    cudaFree(w.z); cudaFree(w.gz); cudaFree(w.S); cudaFree(w.Y); cudaFree(w.sy); cudaFree(w.hcount); cudaFree(w.hhead); cudaFree(w.moved);
    w.z = w.gz = w.S = w.Y = w.sy = nullptr; w.hcount = w.hhead = w.moved = nullptr; w.hist = 0;
    *bytes -= w.lbfgs_bytes;   // a longer history replaces the arrays: their bytes are counted once
    w.lbfgs_bytes = 0;
    const size_t np = (size_t)(nparam > 0 ? nparam : 1) * sizeof(double);
    bool ok = true;
    ok &= cudaMalloc((void **)&w.z, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.gz, np) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.S, np * (hist + 1)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.Y, np * (hist + 1)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.sy, (size_t)batch * (hist + 1) * sizeof(double)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.hcount, (size_t)batch * sizeof(int32_t)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.hhead, (size_t)batch * sizeof(int32_t)) == cudaSuccess;
    ok &= cudaMalloc((void **)&w.moved, (size_t)batch * sizeof(int32_t)) == cudaSuccess;
    if (!ok) {
        cudaFree(w.z); cudaFree(w.gz); cudaFree(w.S); cudaFree(w.Y); cudaFree(w.sy); cudaFree(w.hcount); cudaFree(w.hhead); cudaFree(w.moved);
        w.z = w.gz = w.S = w.Y = w.sy = nullptr; w.hcount = w.hhead = w.moved = nullptr;
        return 1;
    }
    w.hist = hist;
    w.lbfgs_bytes = (int64_t)(np * (2 + 2 * (size_t)(hist + 1)) + (size_t)batch * ((hist + 1) * 8 + 12));
    *bytes += w.lbfgs_bytes;
    return 0;
}

constexpr int OPT_THREADS = 256;

// block-wide reductions over OPT_THREADS threads, deterministic (fixed tree)
__device__ __forceinline__ double block_sum(double v, double *sh) {
    const int tid = threadIdx.x;
    sh[tid] = v;
    __syncthreads();
    for (int s = OPT_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) sh[tid] += sh[tid + s];
        __syncthreads();
    }
    const double r = sh[0];
    __syncthreads();
    return r;
}
// max with lowest-index tie break (want_min: min with lowest index)
__device__ __forceinline__ void block_argbest(double &val, long long &idx, bool want_min, double *shv, long long *shi) {
    const int tid = threadIdx.x;
    shv[tid] = val; shi[tid] = idx;
    __syncthreads();
    for (int s = OPT_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) {
            const double a = shv[tid], b = shv[tid + s];
            const long long ia = shi[tid], ib = shi[tid + s];
            const bool take_b = (ib >= 0) && (ia < 0 || (want_min ? (b < a) : (b > a)) || (b == a && ib < ia));
            if (take_b) { shv[tid] = b; shi[tid] = ib; }
        }
        __syncthreads();
    }
    val = shv[0]; idx = shi[0];
    __syncthreads();
}

// Release score of parameter i (A2, L519-L523 with the sign of the prose, R14): > 0 when the descent direction -g
// points from the bound it sits on into the interior.
__device__ __forceinline__ double release_score(const OptWork &w, int64_t i, double cscale) {
    const int8_t p = w.pivot[i];
    if (p == 0) return 0.0;
    const double gint = cscale * w.grad[i] * (w.hi[i] - w.lo[i]);
    return (p < 0) ? -gint : gint;
}
// The n-th highest positive release score of the entry's parameters [o0, o1) (n >= 2), by an 8-bit radix select on
// the bit patterns (positive doubles order like unsigned integers); 0 when fewer than n scores are positive (then
// every positive score is released).  Integer histograms in shared memory: deterministic.
__device__ __forceinline__ double nth_highest_score(const OptWork &w, int64_t o0, int64_t o1, double cscale, int n, uint32_t *hist,
                                                    unsigned long long *sh_prefix, int *sh_n) {
    const int tid = threadIdx.x;
    unsigned long long prefix = 0ull, mask = 0ull;
    int want = n;
    for (int shift = 56; shift >= 0; shift -= 8) {
        for (int b = tid; b < 256; b += OPT_THREADS) hist[b] = 0u;
        __syncthreads();
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) {
            const double sc = release_score(w, i, cscale);
            if (sc > 0.0) {
                const unsigned long long k = (unsigned long long)__double_as_longlong(sc);
                if ((k & mask) == prefix) atomicAdd(&hist[(unsigned)((k >> shift) & 0xffull)], 1u);
            }
        }
        __syncthreads();
        if (tid == 0) {
            int acc = 0, digit = -1;
            for (int b = 255; b >= 0; --b) {
                if (acc + (int)hist[b] >= want) { digit = b; break; }
                acc += (int)hist[b];
            }
            if (digit < 0) { *sh_n = -1; }                  // fewer than `want` candidates: release every positive score
            else { *sh_n = want - acc; *sh_prefix = prefix | ((unsigned long long)digit << shift); }
        }
        __syncthreads();
        if (*sh_n < 0) return 0.0;
        want = *sh_n;
        prefix = *sh_prefix;
        mask |= 0xffull << shift;
        __syncthreads();
    }
    return __longlong_as_double((long long)prefix);
}

// A1 (L509-L513): map the start into [0,1], set the pivots, clear the AdaBelief moments.
__global__ void k_opt_init(OptWork w, int64_t nparam, const double *params, int32_t batch) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *w.iter = 0;
    if (i < batch) w.cscale[i] = 1.0;
    if (i >= nparam) return;
    const double l = w.lo[i], u = w.hi[i];
    double y = (params[i] - l) / (u - l);
    y = fmin(fmax(y, 0.0), 1.0);
    w.y[i] = y;
    w.pivot[i] = y <= 0.0 ? -1 : (y >= 1.0 ? 1 : 0);
    w.m[i] = 0.0; w.v[i] = 0.0; w.dir[i] = 0.0;
    w.x[i] = l + y * (u - l);
}

// Alg. 1 lines 3-17 for one entry per CTA.
__global__ void __launch_bounds__(OPT_THREADS) k_opt_direction(OptWork w, OptShape sh, OptHyper hy) {
    const int32_t iter = *w.iter;
    __shared__ double shv[OPT_THREADS];
    __shared__ long long shi[OPT_THREADS];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t o0 = sh.param_off[e], o1 = sh.param_off[e + 1];
    double cscale = w.cscale[e];
    // the objective the line search compares is 1/2 chi^2 of the GLS residual (= nll + const, evaluated accurately)
    double L = w.Lcur[e] * cscale;
    // release (A2): the n bound parameters whose descent direction -g points furthest into the interior
    __shared__ uint32_t hist[256];
    __shared__ unsigned long long sh_prefix;
    __shared__ int sh_n;
    int nrel = 1;
    if (hy.topk > 0.0) {
        double nb = 0.0;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) nb += (w.pivot[i] != 0) ? 1.0 : 0.0;
        nb = block_sum(nb, shv);
        nrel = max(1, (int)floor(hy.topk * nb));
    }
    if (nrel == 1) {   // the single highest score, lowest index on ties
        double best = 0.0;
        long long bi = -1;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) {
            const double score = release_score(w, i, cscale);
            if (score > 0.0 && (bi < 0 || score > best)) { best = score; bi = i; }
        }
        block_argbest(best, bi, false, shv, shi);
        if (tid == 0 && bi >= 0) w.pivot[bi] = 0;
    } else {           // every score >= the n-th highest positive one
        const double thr = nth_highest_score(w, o0, o1, cscale, nrel, hist, &sh_prefix, &sh_n);
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) {
            const double score = release_score(w, i, cscale);
            if (score > 0.0 && score >= thr) w.pivot[i] = 0;
        }
    }
    __syncthreads();
    // projected gradient norm and dynamic rescale (A4)
    double n2 = 0.0;
    for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS)
        if (w.pivot[i] == 0) {
            const double gint = cscale * w.grad[i] * (w.hi[i] - w.lo[i]);
            n2 += gint * gint;
        }
    n2 = block_sum(n2, shv);
    const double nrm = sqrt(n2);
    double f = 1.0;
    if (nrm > 0.0 && (nrm < hy.safe_lo || nrm > hy.safe_hi)) f = 1.0 / nrm;
    cscale *= f;
    L *= f;
    // AdaBelief direction, masked; directional derivative; distance to the nearest bound
    const double t = (double)(iter + 1);
    const double bc1 = 1.0 - pow(hy.beta1, t), bc2 = 1.0 - pow(hy.beta2, t);
    double gd = 0.0, amax = CUDART_INF;
    long long il = -1;
    for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) {
        const bool free_i = w.pivot[i] == 0;
        const double g = free_i ? cscale * w.grad[i] * (w.hi[i] - w.lo[i]) : 0.0;
        double m = w.m[i] * f, v = w.v[i] * f * f;
        m = hy.beta1 * m + (1.0 - hy.beta1) * g;
        const double dgm = g - m;
        v = hy.beta2 * v + (1.0 - hy.beta2) * dgm * dgm + hy.eps;
        w.m[i] = m; w.v[i] = v;
        double d = free_i ? -hy.lr * (m / bc1) / (sqrt(v / bc2) + hy.eps) : 0.0;
        w.dir[i] = d;
        gd += g * d;
        if (d != 0.0) {
            const double y = w.y[i];
            const double a = d > 0.0 ? (1.0 - y) / d : y / (-d);
            if (il < 0 || a < amax) { amax = a; il = i; }
        }
    }
    gd = block_sum(gd, shv);
    block_argbest(amax, il, true, shv, shi);
    if (tid == 0) {
        w.cscale[e] = cscale;
        w.L0[e] = L;
        w.gd[e] = gd;
        w.amax[e] = (il >= 0) ? amax : CUDART_INF;
        w.ilim[e] = il;
        w.alpha[e] = (il >= 0) ? fmin(1.0, amax) : 1.0;
        w.alpha_acc[e] = 0.0;
        w.accepted[e] = 0;
    }
}

// trial point x_t = l + clamp(y + alpha d)(u - l); grid = (batch, ceil(ktot_max/256)): the entry on grid.x, which has no 65535 limit
__global__ void k_opt_trial(OptWork w, OptShape sh) {
    const int e = blockIdx.x;
    const int64_t i = sh.param_off[e] + (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= sh.param_off[e + 1]) return;
    const double a = w.accepted[e] ? w.alpha_acc[e] : w.alpha[e];
    const double y = fmin(fmax(w.y[i] + a * w.dir[i], 0.0), 1.0);
    w.xt[i] = w.lo[i] + y * (w.hi[i] - w.lo[i]);
}

// Armijo test per entry (L263: every accepted step decreases the objective)
__global__ void k_opt_ls(OptWork w, OptShape sh, OptHyper hy) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= sh.batch || w.accepted[e]) return;
    double half_chi2 = 0.0;   // nll_reg_t holds chi^2 per region at the trial point
    for (int r = 0; r < sh.nregion; ++r) half_chi2 += w.nll_reg_t[(int64_t)e * sh.nregion + r];
    half_chi2 *= 0.5;
    const double Lt = half_chi2 * w.cscale[e];
    const double a = w.alpha[e];
    // sufficient decrease with min(g.d, 0): a momentum direction with g.d >= 0 never licenses an increase (L263)
    if (Lt <= w.L0[e] + hy.c1 * a * fmin(w.gd[e], 0.0) + hy.ls_noise * fabs(w.L0[e])) {   // false for NaN / +inf
        w.accepted[e] = 1;
        w.alpha_acc[e] = a;
        w.Lt_acc[e] = half_chi2;
    } else {
        w.alpha[e] = 0.5 * a;
    }
}

// lines 19-25: move, pin the limiting parameter if the step reached alpha_max
__global__ void k_opt_commit(OptWork w, OptShape sh) {
    const int e = blockIdx.x;
    if (blockIdx.y == 0 && e == 0 && threadIdx.x == 0) *w.iter += 1;   // k_opt_direction of this iteration is done
    if (blockIdx.y == 0 && threadIdx.x == 0 && w.accepted[e]) w.Lcur[e] = w.Lt_acc[e];
    const int64_t i = sh.param_off[e] + (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= sh.param_off[e + 1]) return;
    const double a = w.accepted[e] ? w.alpha_acc[e] : 0.0;
    double y = fmin(fmax(w.y[i] + a * w.dir[i], 0.0), 1.0);
    if (a > 0.0 && a == w.amax[e] && i == w.ilim[e]) {
        y = w.dir[i] > 0.0 ? 1.0 : 0.0;
        w.pivot[i] = w.dir[i] > 0.0 ? 1 : -1;
    } else if (w.pivot[i] == 0 && a > 0.0 && (y <= 0.0 || y >= 1.0)) {
        w.pivot[i] = y <= 0.0 ? -1 : 1;
    }
    w.y[i] = y;
    w.x[i] = w.lo[i] + y * (w.hi[i] - w.lo[i]);
}

// 1/2 chi^2 at the start point (nll_reg_t holds chi^2 per region there)
__global__ void k_opt_setL(OptWork w, OptShape sh) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= sh.batch) return;
    double c2 = 0.0;
    for (int r = 0; r < sh.nregion; ++r) c2 += w.nll_reg_t[(int64_t)e * sh.nregion + r];
    w.Lcur[e] = 0.5 * c2;
}

__global__ void k_opt_finish(OptWork w, OptShape sh, double *params, double *nll_final) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < sh.nparam) params[i] = w.x[i];
    if (nll_final && i < sh.batch) {
        double L = 0.0;
        for (int r = 0; r < sh.nregion; ++r) L += w.nll_reg[i * sh.nregion + r];
        nll_final[i] = L;
    }
}

// ------------------------------------------------------------------------------------------------------------
// L-BFGS back-end (f4(i); "multiple solvers (L-BFGS, AdaTopK, ...), box constraints via sigmoid
// reparameterisation"; reading R19 of DESIGN.md; Liu & Nocedal 1989, Nocedal & Wright Alg. 7.4 / 7.5).
//   x = l + (u - l) sigma(z);  g_z = g_x (u - l) y (1 - y), y = sigma(z);  d = -H g_z by the two-loop recursion over
//   the stored pairs; backtracking Armijo line search from alpha = 1 on 1/2 chi^2 (the kernels of the AdaTopK line
//   search); pair (s, yv) = (alpha d, g_z+ - g_z) stored when s.yv > curv_eps |s| |yv|.
// ------------------------------------------------------------------------------------------------------------
constexpr int LBFGS_HIST_MAX = 32;
__device__ __forceinline__ double sigmoid_(double z) { return 0.5 * (1.0 + tanh(0.5 * z)); }

__global__ void k_lb_init(OptWork w, int64_t nparam, const double *params, int32_t batch, double ymin) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *w.iter = 0;
    if (i < batch) { w.cscale[i] = 1.0; w.hcount[i] = 0; w.hhead[i] = 0; w.moved[i] = 0; }
    if (i >= nparam) return;
    const double l = w.lo[i], u = w.hi[i];
    double y = (params[i] - l) / (u - l);
    y = fmin(fmax(y, ymin), 1.0 - ymin);
    const double z = log(y) - log1p(-y);
    w.z[i] = z;
    w.gz[i] = 0.0; w.dir[i] = 0.0;
    w.x[i] = l + (u - l) * sigmoid_(z);
}

// One entry per CTA: gradient in z, pair update, two-loop recursion, directional derivative.
__global__ void __launch_bounds__(OPT_THREADS) k_lb_direction(OptWork w, OptShape sh, int32_t hist, double curv_eps) {
    __shared__ double shv[OPT_THREADS];
    __shared__ double s_a[LBFGS_HIST_MAX];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t o0 = sh.param_off[e], o1 = sh.param_off[e + 1], np = sh.nparam;
    const int nslot = hist + 1;   // the new pair is written to the slot after the newest: never one of the <= hist valid ones
    int count = w.hcount[e], head = w.hhead[e];
    const bool moved = w.moved[e] != 0;
    const double a_acc = w.alpha_acc[e];
    // gradient in z at the current point; the new pair (s, yv) = (alpha d, g_z - g_z of the previous point)
    double sy = 0.0, ss = 0.0, yy = 0.0, gg = 0.0;
    for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) {
        const double y = sigmoid_(w.z[i]);
        const double g = w.grad[i] * (w.hi[i] - w.lo[i]) * y * (1.0 - y);
        if (moved) {
            const double s = a_acc * w.dir[i], yv = g - w.gz[i];
            w.S[(int64_t)head * np + i] = s;      // written to the next slot; kept only if the curvature test passes
            w.Y[(int64_t)head * np + i] = yv;
            sy += s * yv; ss += s * s; yy += yv * yv;
        }
        w.gz[i] = g;
        gg += g * g;
    }
    sy = block_sum(sy, shv); ss = block_sum(ss, shv); yy = block_sum(yy, shv); gg = block_sum(gg, shv);
    if (moved) {
        if (sy > curv_eps * sqrt(ss) * sqrt(yy)) {
            if (tid == 0) w.sy[(int64_t)head * sh.batch + e] = sy;
            head = (head + 1) % nslot;
            count = min(count + 1, hist);
        }
    } else {
        count = 0;   // the line search found no step (or this is the first iteration): no history
    }
    __syncthreads();
    // two-loop recursion on q = dir (Nocedal & Wright Alg. 7.4), newest pair first
    for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) w.dir[i] = w.gz[i];
    __syncthreads();
    for (int j = 0; j < count; ++j) {
        const int slot = ((head - 1 - j) % nslot + nslot) % nslot;
        double sq = 0.0;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) sq += w.S[(int64_t)slot * np + i] * w.dir[i];
        sq = block_sum(sq, shv);
        const double a = sq / w.sy[(int64_t)slot * sh.batch + e];
        if (tid == 0) s_a[j] = a;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) w.dir[i] -= a * w.Y[(int64_t)slot * np + i];
        __syncthreads();
    }
    if (count > 0) {   // H0 = gamma I with the newest pair
        const int slot = ((head - 1) % nslot + nslot) % nslot;
        double y2 = 0.0;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) { const double yv = w.Y[(int64_t)slot * np + i]; y2 += yv * yv; }
        y2 = block_sum(y2, shv);
        const double gamma = w.sy[(int64_t)slot * sh.batch + e] / y2;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) w.dir[i] *= gamma;
        __syncthreads();
    }
    for (int j = count - 1; j >= 0; --j) {   // oldest pair first
        const int slot = ((head - 1 - j) % nslot + nslot) % nslot;
        double yr = 0.0;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) yr += w.Y[(int64_t)slot * np + i] * w.dir[i];
        yr = block_sum(yr, shv);
        const double b = yr / w.sy[(int64_t)slot * sh.batch + e];
        const double a = s_a[j];
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) w.dir[i] += w.S[(int64_t)slot * np + i] * (a - b);
        __syncthreads();
    }
    double gd = 0.0;
    for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) { const double d = -w.dir[i]; w.dir[i] = d; gd += w.gz[i] * d; }
    gd = block_sum(gd, shv);
    const double nrm = sqrt(gg);
    if (count == 0 || !(gd < 0.0)) {   // no pair yet, or not a descent direction (rounding): unit steepest-descent step
        count = 0;
        const double inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
        for (int64_t i = o0 + tid; i < o1; i += OPT_THREADS) w.dir[i] = -w.gz[i] * inv;
        gd = -nrm;
    }
    if (tid == 0) {
        w.hcount[e] = count; w.hhead[e] = head;
        w.L0[e] = w.Lcur[e];
        w.gd[e] = gd;
        w.alpha[e] = 1.0;
        w.alpha_acc[e] = 0.0;
        w.accepted[e] = 0;
    }
}

// trial point x_t = l + (u - l) sigma(z + alpha d); grid = (batch, ceil(ktot_max/256)): the entry on grid.x, which has no 65535 limit
__global__ void k_lb_trial(OptWork w, OptShape sh) {
    const int e = blockIdx.x;
    const int64_t i = sh.param_off[e] + (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= sh.param_off[e + 1]) return;
    const double a = w.accepted[e] ? w.alpha_acc[e] : w.alpha[e];
    w.xt[i] = w.lo[i] + (w.hi[i] - w.lo[i]) * sigmoid_(w.z[i] + a * w.dir[i]);
}

__global__ void k_lb_commit(OptWork w, OptShape sh) {
    const int e = blockIdx.x;
    if (blockIdx.y == 0 && e == 0 && threadIdx.x == 0) *w.iter += 1;
    const bool acc = w.accepted[e] != 0;
    if (blockIdx.y == 0 && threadIdx.x == 0) {
        if (acc) w.Lcur[e] = w.Lt_acc[e];
        w.moved[e] = acc ? 1 : 0;
    }
    const int64_t i = sh.param_off[e] + (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= sh.param_off[e + 1] || !acc) return;
    const double z = w.z[i] + w.alpha_acc[e] * w.dir[i];
    w.z[i] = z;
    w.x[i] = w.lo[i] + (w.hi[i] - w.lo[i]) * sigmoid_(z);
}

inline void lb_init(OptWork &w, const OptShape &sh, const double *params, const double *lo, const double *hi, double ymin, cudaStream_t st) {
    w.lo = lo; w.hi = hi;
    const int64_t n = sh.nparam > sh.batch ? sh.nparam : sh.batch;
    k_lb_init<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w, sh.nparam, params, sh.batch, ymin);
}
inline void lb_direction(OptWork &w, const OptShape &sh, int32_t hist, double curv_eps, cudaStream_t st) {
    k_lb_direction<<<sh.batch, OPT_THREADS, 0, st>>>(w, sh, hist, curv_eps);
}
inline void lb_trial_point(OptWork &w, const OptShape &sh, cudaStream_t st) {
    dim3 grid(sh.batch, (sh.ktot_max + 255) / 256);
    k_lb_trial<<<grid, 256, 0, st>>>(w, sh);
}
inline void lb_commit(OptWork &w, const OptShape &sh, cudaStream_t st) {
    dim3 grid(sh.batch, (sh.ktot_max + 255) / 256);
    k_lb_commit<<<grid, 256, 0, st>>>(w, sh);
}

inline void opt_init(OptWork &w, const OptShape &sh, const double *params, const double *lo, const double *hi, cudaStream_t st) {
    w.lo = lo; w.hi = hi;
    const int64_t n = sh.nparam > sh.batch ? sh.nparam : sh.batch;
    k_opt_init<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w, sh.nparam, params, sh.batch);
}
inline void opt_direction(OptWork &w, const OptShape &sh, const OptHyper &hy, cudaStream_t st) {
    k_opt_direction<<<sh.batch, OPT_THREADS, 0, st>>>(w, sh, hy);
}
inline void opt_trial_point(OptWork &w, const OptShape &sh, cudaStream_t st) {
    dim3 grid(sh.batch, (sh.ktot_max + 255) / 256);
    k_opt_trial<<<grid, 256, 0, st>>>(w, sh);
}
inline void opt_ls_update(OptWork &w, const OptShape &sh, const OptHyper &hy, cudaStream_t st) {
    k_opt_ls<<<(sh.batch + 127) / 128, 128, 0, st>>>(w, sh, hy);
}
inline void opt_set_L(OptWork &w, const OptShape &sh, cudaStream_t st) {
    k_opt_setL<<<(sh.batch + 127) / 128, 128, 0, st>>>(w, sh);
}
inline void opt_commit(OptWork &w, const OptShape &sh, cudaStream_t st) {
    dim3 grid(sh.batch, (sh.ktot_max + 255) / 256);
    k_opt_commit<<<grid, 256, 0, st>>>(w, sh);
}
inline void opt_finish(OptWork &w, const OptShape &sh, double *params, double *nll_final, cudaStream_t st) {
    const int64_t n = sh.nparam > sh.batch ? sh.nparam : sh.batch;
    k_opt_finish<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w, sh, params, nll_final);
}

}  // namespace cs
