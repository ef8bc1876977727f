// cs_kmeans.cuh -- f2: batched spherical K-means patching, the step right before the hot path.
//
// Pixels are unit vectors n_p; a patch is the set of pixels closest (largest dot product, L100-L102) to a centroid;
// a Lloyd iteration moves every centroid to the renormalised mean of its pixels (L104).  Many independent problems
// (one per spectral parameter, patch count and sky region) run in one launch each step.
//
// Index work must be bit-exact, so the arithmetic is pinned down rather than left to the compiler:
//   dot      = (x * cx + y * cy) + z * cz, every operation rounded once (no FMA)       fp64
//   argmax   : ties to the lowest patch id
//   sums[k]  = sum of n_p over the patch's pixels in ascending pixel order, one fp64 add at a time
//   centroid = sums / sqrt((sx*sx + sy*sy) + sz*sz) ; an empty patch keeps its centroid (and its label)
// The dot products are a [npix,3] x [3,K] contraction: three multiply-adds per output, HBM- and latency-trivial, no
// shared operand worth a tensor-core tile.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cs {

struct KmProb {
    int32_t K;         // patches of this problem (>= 1)
    int32_t region;    // -1: every pixel takes part; else only the pixels with region[p] == region
    int64_t coff;      // first centroid of the problem in the centroid array
};

constexpr int KM_TILE = 1024;   // centroids staged in shared memory at a time

// labels[j][p] = argmax_k n_p . c_k (or -1 outside the problem's region).  grid = (ceil(npix/256), nprob), block = 256.
__global__ void __launch_bounds__(256) k_km_assign(const double *__restrict__ vecs, int64_t npix, const uint8_t *__restrict__ region,
                                                   const KmProb *__restrict__ probs, const double *__restrict__ cent,
                                                   int32_t *__restrict__ labels) {
    __shared__ double sc[KM_TILE * 3];
    const KmProb pr = probs[blockIdx.y];
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = p < npix && (pr.region < 0 || region[p] == pr.region);
    double x = 0, y = 0, z = 0;
    if (in) { x = vecs[3 * p]; y = vecs[3 * p + 1]; z = vecs[3 * p + 2]; }
    double best = -2.0;
    int bk = 0;
    for (int k0 = 0; k0 < pr.K; k0 += KM_TILE) {
        const int nk = min(KM_TILE, pr.K - k0);
        __syncthreads();
        for (int i = threadIdx.x; i < 3 * nk; i += blockDim.x) sc[i] = cent[3 * (pr.coff + k0) + i];
        __syncthreads();
        if (in)
            for (int k = 0; k < nk; ++k) {
                const double dot = __dadd_rn(__dadd_rn(__dmul_rn(x, sc[3 * k]), __dmul_rn(y, sc[3 * k + 1])), __dmul_rn(z, sc[3 * k + 2]));
                if (dot > best) { best = dot; bk = k0 + k; }   // strict: ties keep the lower id
            }
    }
    if (p < npix) labels[(int64_t)blockIdx.y * npix + p] = in ? bk : -1;
}

// Centroid update: warp = one patch, block = eight patches.  The block walks the labels in chunks staged in shared
// memory.  Per chunk a warp first compacts the positions of its patch's pixels into its own list (ballot + popc, so the
// list is in ascending pixel order), then takes the list 32 entries at a time: the lanes gather the vectors (one load
// latency per 32 pixels), park them in shared memory, and every lane adds them one after the other -- the same sequence
// of fp64 additions as in the generator, one add at a time.
// (Measured, Lloyd iteration of the 30 problems of the clustering scan, against 0.16 ms for the assignment: one thread
// per patch walking all labels 4.35 ms; hits handed over by shuffle straight from the scan 2.35 ms, the K = 5 problem
// alone 2 ms: three dependent shuffle + add pairs and an exposed gather per 32 labels.)
// grid = (ceil(Kmax/8), nprob), block = 256.
constexpr int KM_CHUNK = 2048;
__global__ void __launch_bounds__(256) k_km_update(const double *__restrict__ vecs, int64_t npix, const KmProb *__restrict__ probs,
                                                   const int32_t *__restrict__ labels, double *__restrict__ cent) {
    __shared__ int32_t sl[KM_CHUNK];
    __shared__ uint16_t slist[8][KM_CHUNK];
    __shared__ double sbuf[8][3][32];
    const KmProb pr = probs[blockIdx.y];
    if ((int)(blockIdx.x * 8) >= pr.K) return;   // block-uniform
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int k = blockIdx.x * 8 + warp;
    const bool mine = k < pr.K;                  // warp-uniform
    const int32_t *lab = labels + (int64_t)blockIdx.y * npix;
    const unsigned lt = (1u << lane) - 1u;
    double sx = 0, sy = 0, sz = 0;
    for (int64_t p0 = 0; p0 < npix; p0 += KM_CHUNK) {
        const int n = (int)min((int64_t)KM_CHUNK, npix - p0);
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) sl[i] = lab[p0 + i];
        __syncthreads();
        if (!mine) continue;
        int cnt = 0;
#pragma unroll 4
        for (int i0 = 0; i0 < n; i0 += 32) {
            const int i = i0 + lane;
            const bool hit = i < n && sl[i] == k;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) slist[warp][cnt + __popc(m & lt)] = (uint16_t)i;
            cnt += __popc(m);
        }
        __syncwarp();
        for (int b0 = 0; b0 < cnt; b0 += 32) {
            const int nb = min(32, cnt - b0);
            if (lane < nb) {
                const double *v = vecs + 3 * (p0 + slist[warp][b0 + lane]);
                sbuf[warp][0][lane] = v[0]; sbuf[warp][1][lane] = v[1]; sbuf[warp][2][lane] = v[2];
            }
            __syncwarp();
#pragma unroll 4
            for (int c = 0; c < nb; ++c) {
                sx = __dadd_rn(sx, sbuf[warp][0][c]);
                sy = __dadd_rn(sy, sbuf[warp][1][c]);
                sz = __dadd_rn(sz, sbuf[warp][2][c]);
            }
            __syncwarp();
        }
    }
    if (mine && lane == 0) {
        const double nrm = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(sx, sx), __dmul_rn(sy, sy)), __dmul_rn(sz, sz)));
        if (nrm > 0.0) {
            double *c = cent + 3 * (pr.coff + k);
            c[0] = __ddiv_rn(sx, nrm); c[1] = __ddiv_rn(sy, nrm); c[2] = __ddiv_rn(sz, nrm);
        }
    }
}

}  // namespace cs
