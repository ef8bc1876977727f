// cs_pipe.cuh -- what the two fused kernels share besides the arithmetic: launch parameters, mbarrier / bulk-copy /
// TMA helpers (PTX ISA: mbarrier, cp.async.bulk, cp.async.bulk.tensor), the walk of a CTA over its share of the
// work, and the data loader.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"

namespace cs {

constexpr int MODE_VALUE = 0;   // ll only
constexpr int MODE_GRAD = 1;    // ll + three gradient terms
constexpr int MODE_MAPS = 2;    // component maps (direct kernel, in-place layout)
constexpr int MODE_CMBVAR = 3;  // sums for the CMB-variance metric (Eq. 10)
constexpr int MODE_CHI2 = 4;    // chi^2 of the GLS residual per region (accurate objective differences for the line search)
template <int MODE>
struct ModeTraits {
    static constexpr bool region_only = (MODE == MODE_VALUE || MODE == MODE_CHI2);   // only term 3 is reduced
    static constexpr bool grad = (MODE == MODE_GRAD);
    static constexpr bool reduce = (MODE != MODE_MAPS);
};

struct LikeParams {
    const float *d;            // caller's data [ndata][2*nfreq][npix]
    int64_t npix;
    int32_t nfreq;
    int32_t use_tma;           // 1: rows of d are 16-byte aligned -> tensor-map loads; 0: plain loads
    int32_t evict_first;       // 1: the stream is much larger than L2 and read once -> L2 evict-first policy
    int32_t ring_maps;         // 1: use the pixel-space maps (rmap) and the caller's d whatever the layout (MODE_MAPS)
    const float *dcopy;        // private sorted copies
    const PosInfo *pinfo;      // [entries of the launch's list] table block and data source of the entry at each position
    const MapDev *maps;
    const CfgDev *cfgs;
    const Run *runs;
    int32_t nrun;
    int32_t maps_planes;       // MODE_MAPS: 6 = all components (cmb, dust, sync) x (Q, U); 2 = the CMB component only
    int64_t W;                 // total units of the launch
    const int32_t *elist;
    const int32_t *skip;       // [batch] or null: entries with a non-zero flag are left out (line-search trials of
                               // entries that already accepted a step); their outputs keep their previous values
    const float *tab;
    double *partial;
    int64_t PS;                // doubles per partial row
    float *maps_out;           // MODE_MAPS: [nsel,3,2,npix]
    int32_t *err;
    const double *pcopy;       // copy of the parameters the tables were built from (per-pixel beta_d path)
    float cdf[NROW], l2h[NROW], l2l[NROW];   // cd[f] and log2(nu_f/nu0d) as a float pair (per-pixel beta_d path)
    KConst kc;
};

// ----------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// global -> shared bulk copy completing on an mbarrier; dst/src/bytes 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tma_box_g2s(void *dst, const CUtensorMap *map, int x, int y, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
// Pulls the 64-byte table row at p towards L1 (no register is tied up while it is in flight).
__device__ __forceinline__ void prefetch_row(const float *p) {
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p + 8));
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_normal() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// Named-barrier hand-over (bar.arrive by the producers, bar.sync by the consumer of the hand-over): a warp blocked in
// bar.sync takes no issue slots, unlike a polling mbarrier wait.
__device__ __forceinline__ void named_arrive(int id, int count) {
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void named_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// ----------------------------------------------------------------------------------------------------------
// The walk of a CTA over its share of the launch.  The units of all runs are numbered consecutively (run-major,
// then tile, then entry); CTA b of G takes the units [W b / G, W (b+1) / G): a perfectly balanced, static partition
// (every unit costs the same), in which a CTA changes tile a handful of times over the whole launch.  Every role
// of a CTA walks the same sequence and counts the same live (not skipped) entries, so ring slots and barrier
// phases agree without any communication.
// ----------------------------------------------------------------------------------------------------------
struct Walk {
    int64_t u, u1;      // next unit, end of this CTA's share
    int32_t r;          // current run
    int32_t tile, k, kend;   // current piece: entries [k, kend) of run r on `tile`
    Run run;
};
__device__ __forceinline__ void walk_init(Walk &w, const LikeParams &P) {
    const int64_t G = gridDim.x, b = blockIdx.x;
    w.u = P.W * b / G;
    w.u1 = P.W * (b + 1) / G;
    int lo = 0, hi = P.nrun - 1;   // last run with ustart <= u
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (P.runs[mid].ustart <= w.u) lo = mid; else hi = mid - 1;
    }
    w.r = lo;
    w.run = P.runs[lo];
    w.tile = -1; w.k = 0; w.kend = 0;
}
// Advances to the next piece (a tile and a range of entries of one run); false when the share is exhausted.
__device__ __forceinline__ bool walk_next(Walk &w, const LikeParams &P) {
    if (w.u >= w.u1) return false;
    while (w.u >= w.run.ustart + (int64_t)w.run.ntile * w.run.count) w.run = P.runs[++w.r];
    const int64_t local = w.u - w.run.ustart;
    w.tile = (int32_t)(local / w.run.count);
    w.k = (int32_t)(local - (int64_t)w.tile * w.run.count);
    const int64_t left = w.u1 - w.u;
    w.kend = (int32_t)((left < (int64_t)(w.run.count - w.k)) ? (int64_t)w.k + left : (int64_t)w.run.count);
    w.u += w.kend - w.k;
    return true;
}

// ----------------------------------------------------------------------------------------------------------
// Loader warp: streams one stage per live entry into the data ring.  A stage holds the tile as two halves of
// [2*nfreq rows][256 positions] fp32.  Sorted layout: one contiguous bulk copy from the entry's private copy.
// In place: two TMA boxes of the caller's d viewed as [ndata*2*nfreq rows, npix] (columns beyond npix read as zero),
// or plain loads by the whole warp when rows of d are not 16-byte aligned.
// ----------------------------------------------------------------------------------------------------------
template <int NF, int ND>
__device__ __forceinline__ void loader_loop(const CUtensorMap *tmap, const LikeParams &P, float *ring, uint64_t *full_d,
                                            uint64_t *empty_d, int lane) {
    constexpr int STAGE = 2 * NF * TPX;   // floats per stage
    const int nrows = 2 * P.nfreq;
    const uint64_t policy = P.evict_first ? policy_evict_first() : policy_evict_normal();
    Walk w;
    walk_init(w, P);
    int n = 0;   // live entries so far
    while (walk_next(w, P)) {
        const CfgDev *cf = P.cfgs + w.run.cfg;
        const bool sorted = cf->sorted && !P.ring_maps;
        for (int k = w.k; k < w.kend; ++k) {
            const int64_t srcinfo = __ldg(&P.pinfo[w.run.estart + k].src);
            if (P.skip && __ldg(P.skip + __ldg(P.elist + w.run.estart + k)) != 0) continue;
            const int s = n % ND;
            float *dst = ring + s * STAGE;
            if (sorted) {
                if (lane == 0) {
                    mbar_wait(&empty_d[s], (uint32_t)(((n / ND) & 1) ^ 1));
                    const uint32_t bytes = (uint32_t)nrows * TPX * 4u;
                    mbar_expect_tx(&full_d[s], bytes);
                    if (NF * 2 == nrows) {
                        bulk_g2s(dst, P.dcopy + srcinfo + (int64_t)w.tile * w.run.tstride, bytes, &full_d[s], policy);
                    } else {   // generic band count: the stage keeps 2*NF rows per half, the copy only 2*nfreq
                        const float *src = P.dcopy + srcinfo + (int64_t)w.tile * w.run.tstride;
                        bulk_g2s(dst, src, bytes / 2, &full_d[s], policy);
                        bulk_g2s(dst + NF * 2 * HALF, src + nrows * HALF, bytes / 2, &full_d[s], policy);
                    }
                }
            } else if (P.use_tma) {
                if (lane == 0) {
                    mbar_wait(&empty_d[s], (uint32_t)(((n / ND) & 1) ^ 1));
                    mbar_expect_tx(&full_d[s], (uint32_t)nrows * TPX * 4u);
                    const int y = (int)srcinfo * nrows;
                    tma_box_g2s(dst, tmap, w.tile * TPX, y, &full_d[s], policy);
                    tma_box_g2s(dst + NF * 2 * HALF, tmap, w.tile * TPX + HALF, y, &full_d[s], policy);
                }
            } else {   // rows of d not 16-byte aligned: plain loads by the whole warp
                mbar_wait(&empty_d[s], (uint32_t)(((n / ND) & 1) ^ 1));
                const int64_t row0 = srcinfo * nrows;
                for (int h = 0; h < 2; ++h)
                    for (int r = 0; r < nrows; ++r)
                        for (int x = lane; x < HALF; x += 32) {
                            const int64_t px = (int64_t)w.tile * TPX + h * HALF + x;
                            dst[(h * NF * 2 + r) * HALF + x] = (px < P.npix) ? P.d[(row0 + r) * P.npix + px] : 0.f;
                        }
                __syncwarp();
                if (lane == 0) mbar_arrive(&full_d[s]);
            }
            ++n;
        }
    }
}

}  // namespace cs
