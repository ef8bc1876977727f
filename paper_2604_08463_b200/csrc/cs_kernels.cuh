// cs_kernels.cuh -- the CUDA kernels of libcs (sm_100a).
//
//   k_tables   a1  SED factor tables, fp64 math -> fp32 rows                     (Eq. 2)
//   k_like     a2  fused per-pixel gather / assemble A / 3x3 solve / likelihood and gradient terms, data streamed
//                  through a cp.async.bulk (TMA) + mbarrier ring, followed in the same CTA by the first level of
//              a3  the ordered fp64 segmented reduction (per-tile segments)        (Eq. 5, 6, 17)
//              a4  (MODE_MAPS) GLS component maps                                 (Eq. 5 / 8)
//   k_merge    a3  second level: fixed-order sum of per-tile partials onto clusters and regions
//
// One thread owns one pixel of a 256-pixel tile and walks over the entries of its group (same clustering
// configuration, different data sets / parameters), so cluster ids, slot ids and the reduction plan are loaded
// once per CTA.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <math_constants.h>
#include "cs_internal.h"
#include "cs_math.cuh"

namespace cs {

constexpr int MODE_VALUE = 0;   // ll only (line search)
constexpr int MODE_GRAD = 1;    // ll + three gradient terms
constexpr int MODE_MAPS = 2;    // component maps
constexpr int MODE_CMBVAR = 3;  // sums for the CMB-variance metric (Eq. 10)
constexpr int MODE_CHI2 = 4;    // chi^2 of the GLS residual per region (accurate objective differences for the line search)
template <int MODE>
struct ModeTraits {
    static constexpr bool region_only = (MODE == MODE_VALUE || MODE == MODE_CHI2);   // only term 3 is reduced
};

constexpr int NST = 2;   // stages of each warp's data ring (both in flight while the warp computes)
constexpr int EC = 4;    // entries buffered between reduce phases

struct LikeParams {
    const float *d;
    int64_t npix;
    int32_t nfreq;
    int32_t use_bulk;          // 1: d is TMA-addressable (16-byte aligned rows) -> tensor-map loads; 0: plain loads
    int32_t evict_first;       // 1: d is much larger than L2 and streamed once -> L2 evict-first policy
    const MapDev *maps;
    const CfgDev *cfgs;
    const Group *groups;
    const int32_t *elist;
    const int32_t *data_of;
    const int32_t *skip;       // [batch] or null: entries with a non-zero flag are left out (line-search trials of
                               // entries that already accepted a step); their outputs keep their previous values
    const int64_t *tab_off;    // [batch] first table row of entry
    const float *tab;
    double *partial;
    int64_t PS;                // doubles per partial row
    float *maps_out;           // MODE_MAPS: [nsel,3,2,npix], slot = position in elist
    int32_t *err;
    KConst kc;
};

// ----------------------------------------------------------------------------------------------------------
// mbarrier / bulk-copy helpers (PTX ISA: mbarrier, cp.async.bulk)
// ----------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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
// Wait used by producer roles (loader, builders): they are ahead of the consumers most of the time, so the poll
// backs off (suspend hint + nanosleep) instead of burning issue slots the consumers need.
__device__ __forceinline__ void mbar_wait_relaxed(uint64_t *bar, uint32_t parity, unsigned sleep_ns = 40) {
    uint32_t done = 0;
    while (true) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity), "r"(500u)
            : "memory");
        if (done) break;
        __nanosleep(sleep_ns);
    }
}
// global -> shared bulk copy completing on an mbarrier; dst/src/bytes 16-byte aligned; evict-first L2 policy.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
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

// ----------------------------------------------------------------------------------------------------------
// a1: SED factor tables.  One thread per (entry, parameter, band quad).  fp64 -> fp32.
// ----------------------------------------------------------------------------------------------------------
// exp(y) in fp64 for the power-law rows: y = k ln2 + r, |r| <= ln2/2, degree-11 Taylor polynomial (truncation
// 6e-15 relative, far below the fp32 rounding of the stored value), scaled by 2^k through the exponent field.
// Arguments outside the range where 2^k is a normal number take the library routine.
__device__ __forceinline__ double exp_pow(double y) {
    if (!(fabs(y) < 700.0)) return exp(y);
    const double kf = rint(y * 1.4426950408889634074);
    double r = fma(-kf, 6.93147180369123816490e-01, y);
    r = fma(-kf, 1.90821492927058770002e-10, r);
    double p = 1.0 / 39916800.0;
    p = fma(p, r, 1.0 / 3628800.0); p = fma(p, r, 1.0 / 362880.0); p = fma(p, r, 1.0 / 40320.0);
    p = fma(p, r, 1.0 / 5040.0);    p = fma(p, r, 1.0 / 720.0);    p = fma(p, r, 1.0 / 120.0);
    p = fma(p, r, 1.0 / 24.0);      p = fma(p, r, 1.0 / 6.0);      p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);             p = fma(p, r, 1.0);
    return p * __hiloint2double(((int)kf + 1023) << 20, 0);
}

// One thread per (entry, parameter, band quad): four table values, one 16-byte store.  The band constants come from a
// shared-memory copy (indexed by the thread's quad: a constant-bank read would serialise).
// grid = (ceil(4 * ktot_max / 256), batch), block = 256.
__global__ void __launch_bounds__(256) k_tables(const double *__restrict__ params, const int64_t *__restrict__ param_off,
                                                const int64_t *__restrict__ tab_off, const int32_t *__restrict__ cfg_of,
                                                const CfgDev *__restrict__ cfgs, float *__restrict__ tab, int32_t batch,
                                                int32_t *err, const TConst *__restrict__ tcg, const int32_t *__restrict__ skip) {
    __shared__ TConst tc;
    for (int i = threadIdx.x; i < (int)(sizeof(TConst) / 8); i += blockDim.x)
        reinterpret_cast<double *>(&tc)[i] = reinterpret_cast<const double *>(tcg)[i];
    __syncthreads();
    const int nfreq = tc.nfreq;
    for (int e = blockIdx.y; e < batch; e += gridDim.y) {
        if (skip && skip[e] != 0) continue;
        const CfgDev *cp = cfgs + cfg_of[e];
        const int K0 = cp->K[0], K1 = cp->K[1], ktot = cp->ktot;
        const int id = blockIdx.x * blockDim.x + threadIdx.x;
        const int j = id >> 2, f0 = (id & 3) * 4;
        if (j >= ktot) continue;
        const double x = params[param_off[e] + j];
        float *row0 = tab + tab_off[e] * NROW;
        bool bad = !isfinite(x);
        float v[4];
        if (j < K0) {
            // dust power-law factor with the band constant folded in: cd[f] * (nu_f/nu0d)^beta_d
#pragma unroll
            for (int i = 0; i < 4; ++i) v[i] = (f0 + i < nfreq) ? (float)(tc.cd[f0 + i] * exp_pow(x * tc.lnd[f0 + i])) : 0.f;
            *reinterpret_cast<float4 *>(row0 + (int64_t)j * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
        } else if (j < K0 + K1) {
            // Planck ratio G = expm1(x0)/expm1(x) and d ln G / dT = (1/T) [ x/(1-e^-x) - x0/(1-e^-x0) ]
            bad = bad || !(x > 0.0);
            const int k = j - K0;
            float dg[4];
            const double x0 = tc.hk * tc.nu0d / x, e0 = expm1(x0), h0 = x0 / (-expm1(-x0));
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                v[i] = 0.f; dg[i] = 0.f;
                if (f0 + i < nfreq) {
                    const double xf = tc.hk * tc.nu[f0 + i] / x;
                    v[i] = (float)(e0 / expm1(xf));
                    dg[i] = (float)((xf / (-expm1(-xf)) - h0) / x);
                }
            }
            *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + k) * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + K1 + k) * NROW + f0) = make_float4(dg[0], dg[1], dg[2], dg[3]);
        } else {
            const int k = j - K0 - K1;
#pragma unroll
            for (int i = 0; i < 4; ++i) v[i] = (f0 + i < nfreq) ? (float)(tc.cs[f0 + i] * exp_pow(x * tc.lns[f0 + i])) : 0.f;
            *reinterpret_cast<float4 *>(row0 + (int64_t)(K0 + 2 * K1 + k) * NROW + f0) = make_float4(v[0], v[1], v[2], v[3]);
        }
        if (bad && f0 == 0) atomicOr(err, ERR_DOMAIN);
    }
}

// ----------------------------------------------------------------------------------------------------------
// a2: per-pixel arithmetic in packed fp32x2 (FFMA2 / FMUL2 / FADD2 on sm_100): the two lanes of every packed
// operation are two consecutive bands (f, f+1), so table rows (float4 loads), constants and data pair up without
// any broadcast; the 16th band is a zero pad.  Accumulators are reduced lane-to-scalar once per pixel.
// ----------------------------------------------------------------------------------------------------------
constexpr int NPAIR = NROW / 2;

// The pixel's data in the warp's shared-memory stage: rows are (band, Stokes), 32 pixels per row.  Both passes
// (forward and gradient) read it from there instead of keeping 30 values in registers.
template <int NF>
struct PixelIn {
    const float *st;   // stage base + lane
    __device__ __forceinline__ float2 dq(int j) const {
        return make_float2(st[(4 * j + 0) * 32], (2 * j + 1 < NF) ? st[(4 * j + 2) * 32] : 0.f);
    }
    __device__ __forceinline__ float2 du(int j) const {
        return make_float2(st[(4 * j + 1) * 32], (2 * j + 1 < NF) ? st[(4 * j + 3) * 32] : 0.f);
    }
};

// ----------------------------------------------------------------------------------------------------------
// a2 + first level of a3: the fused kernel.  grid = (ntile, ngroup), block = TP threads = 8 warps.
//
// Data path: every warp owns the 32 pixels [tile*256 + 32*warp, +32) and streams its own [2*nfreq x 32] box of d
// per entry through a private NST-stage ring filled by TMA (cp.async.bulk.tensor.2d, one instruction per warp and
// entry, completion on the warp's own mbarrier).  Warps never synchronise with each other on the data path.
// Reduction: each thread stores its four terms at the rank its pixel has in the tile's (cluster, pixel) order, so
// that every segment is a contiguous run in shared memory; every EC entries the CTA sums the segments (one thread
// per (entry, term, segment), ascending pixel order, fp64) into the partial buffer.  The term buffer is double
// buffered: one __syncthreads per EC entries.
// shared memory: ring [8 warps][NST][2*NF][32] fp32 | terms [2][EC][4][TP] fp32 | barriers [8][NST] | meta
// (configurations whose tiles hold few distinct cluster triples run on k_like_cell, cs_like_cell.cuh, instead)
// ----------------------------------------------------------------------------------------------------------
constexpr int NWARP = TP / 32;
constexpr int TROW = TP + 4;   // floats per term row: TP ranks + a dump slot for pixels without a rank

// Loads the tile's segment descriptors and output slots of the four reducing maps into shared memory.
// meta[t] = number of segments of term t in this tile (0 for terms below T0).
template <int MODE>
__device__ __forceinline__ void load_tile_plan(const MapDev *__restrict__ maps, const CfgDev &cfg, int tile, int tid,
                                               uint16_t *s_desc, int32_t *s_slot, int32_t *meta) {
    constexpr int T0 = ModeTraits<MODE>::region_only ? 3 : 0;
    if (tid < 4) {
        const int t = tid;
        const int mi = (MODE == MODE_CMBVAR) ? cfg.map[3] : cfg.map[t];
        meta[t] = (t >= T0) ? (maps[mi].segptr[tile + 1] - maps[mi].segptr[tile]) : 0;
    }
#pragma unroll
    for (int t = T0; t < 4; ++t) {
        const int mi = (MODE == MODE_CMBVAR) ? cfg.map[3] : cfg.map[t];
        const int s0 = maps[mi].segptr[tile], s1 = maps[mi].segptr[tile + 1];
        if (tid < s1 - s0) {
            s_desc[t * TP + tid] = maps[mi].segdesc[s0 + tid];
            s_slot[t * TP + tid] = ((MODE == MODE_CMBVAR) ? t * maps[mi].nseg : cfg.segbase[t]) + maps[mi].segslot[s0 + tid];
        }
    }
}

// First level of the ordered reduction (a3) for `nent` buffered entries: one thread per (entry, term, segment); a
// segment is a contiguous run of the rank-ordered terms of one cluster, summed in fp64 in the fixed chunk order of
// cs_math.cuh (the same order as the reducer warps of k_like_cell) and stored at the segment's cluster-major slot of
// the entry's partial row.
__device__ __forceinline__ void reduce_terms(const float *tbuf, int nent, int tid, const int32_t *meta, const uint16_t *s_desc,
                                             const int32_t *s_slot, const int32_t *s_ent, double *__restrict__ partial, int64_t PS) {
    const int n0 = meta[0], n1 = meta[1], n2 = meta[2], n3 = meta[3];
    const int c1 = n0, c2 = n0 + n1, c3 = n0 + n1 + n2, tot = c3 + n3;
    const float inv_tot = 1.0f / (float)tot;
    for (int w = tid; w < nent * tot; w += TP) {
        const int ent = (int)(((float)w + 0.5f) * inv_tot), r = w - ent * tot;
        const int t = (r >= c1) + (r >= c2) + (r >= c3);
        const int ls = r - (t == 0 ? 0 : (t == 1 ? c1 : (t == 2 ? c2 : c3)));
        const uint32_t desc = s_desc[t * TP + ls];
        const int start = desc & 0xff, len = (int)(desc >> 8) + 1;
        partial[(int64_t)s_ent[ent] * PS + s_slot[t * TP + ls]] = segment_sum(tbuf + (ent * 4 + t) * TROW, start, len);
    }
}

template <int NF>
constexpr size_t like_smem_bytes() {
    return (size_t)NWARP * NST * 2 * NF * 32 * 4      // data ring
           + (size_t)2 * EC * 4 * TROW * 4            // double-buffered terms
           + NWARP * NST * 8                          // mbarriers
           + GROUP_MAX * 16                           // per-entry table base (8 B), data row (4 B), entry id (4 B)
           + 4 * TP * 2                               // segment descriptors of the tile, four maps
           + 4 * TP * 4                               // output slots of those segments
           + 16 * 4;                                  // meta
}

__device__ __forceinline__ void tma_box_g2s(void *dst, const CUtensorMap *map, int x, int y, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

// Per-entry arrays of a group in shared memory (table base, first data row, entry id).  With a skip mask the kept
// entries are compacted in order; s_cnt[0] + s_cnt[1] is their number once the caller has synchronised the CTA.
// Called by all threads of the CTA (contains a __syncthreads).
static_assert(GROUP_MAX <= 64, "two warps compact a group");
__device__ __forceinline__ void load_group(const LikeParams &P, const Group &grp, int nrows, int tid, const float **s_tab,
                                           int32_t *s_drow, int32_t *s_ent, int32_t *s_cnt) {
    int e = 0, pos = 0;
    bool keep = false;
    if (tid < 64) {
        if (tid < grp.count) {
            e = P.elist[grp.start + tid];
            keep = !(P.skip && P.skip[e] != 0);
        }
        const unsigned b = __ballot_sync(0xffffffffu, keep);
        pos = __popc(b & ((1u << (tid & 31)) - 1u));
        if ((tid & 31) == 0) s_cnt[tid >> 5] = __popc(b);
    }
    __syncthreads();
    if (keep) {
        if (tid >= 32) pos += s_cnt[0];
        s_ent[pos] = e;
        s_drow[pos] = P.data_of[e] * nrows;
        s_tab[pos] = P.tab + P.tab_off[e] * NROW;
    }
}

template <int NF, int MODE>
__global__ void __launch_bounds__(TP, 2) k_like(const __grid_constant__ CUtensorMap tmap, const LikeParams P) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *sterm = ring + NWARP * NST * 2 * NF * 32;
    uint64_t *bars = reinterpret_cast<uint64_t *>(sterm + 2 * EC * 4 * TROW);
    const float **s_tab = reinterpret_cast<const float **>(bars + NWARP * NST);   // [GROUP_MAX] table base of entry
    int32_t *s_drow = reinterpret_cast<int32_t *>(s_tab + GROUP_MAX);             // [GROUP_MAX] first d row of entry
    int32_t *s_ent = s_drow + GROUP_MAX;                                          // [GROUP_MAX] entry id
    uint16_t *s_desc = reinterpret_cast<uint16_t *>(s_ent + GROUP_MAX);           // [4][TP] segment descriptors
    int32_t *s_slot = reinterpret_cast<int32_t *>(s_desc + 4 * TP);               // [4][TP] output slots
    int32_t *meta = s_slot + 4 * TP;                                              // [0..3] segments per term

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x;
    const Group grp = P.groups[blockIdx.y];
    const CfgDev cfg = P.cfgs[grp.cfg];
    const int64_t npix = P.npix;
    const int64_t p = (int64_t)tile * TP + tid;
    const int nrows = 2 * P.nfreq;
    constexpr bool kReduce = (MODE != MODE_MAPS);
    int k0 = -1, k1 = -1, k2 = -1;
    // float offset of this pixel's slot in each term row: its rank in the tile's (cluster, pixel) order of the
    // reducing map, or the dump slot TP when the pixel has no cluster there
    int so0 = 0 * TROW + TP, so1 = 1 * TROW + TP, so2 = 2 * TROW + TP, so3 = 3 * TROW + TP;
    if (p < npix) {
        k0 = P.maps[cfg.map[0]].idx[p];
        k1 = P.maps[cfg.map[1]].idx[p];
        k2 = P.maps[cfg.map[2]].idx[p];
        if (kReduce) {
            const int m3 = cfg.map[3];
            if (MODE == MODE_CMBVAR) {
                const int r = P.maps[m3].rank[p];
                so0 = 0 * TROW + r; so1 = 1 * TROW + r; so2 = 2 * TROW + r; so3 = 3 * TROW + r;
            } else {
                if (!ModeTraits<MODE>::region_only) {
                    if (k0 >= 0) so0 = 0 * TROW + P.maps[cfg.map[0]].rank[p];
                    if (k1 >= 0) so1 = 1 * TROW + P.maps[cfg.map[1]].rank[p];
                    if (k2 >= 0) so2 = 2 * TROW + P.maps[cfg.map[2]].rank[p];
                }
                so3 = 3 * TROW + P.maps[m3].rank[p];
            }
        }
    }
    const bool live = (k0 >= 0) && (k1 >= 0) && (k2 >= 0);
    if (kReduce) load_tile_plan<MODE>(P.maps, cfg, tile, tid, s_desc, s_slot, meta);
    load_group(P, grp, nrows, tid, s_tab, s_drow, s_ent, meta + 12);
    float *wring = ring + warp * NST * 2 * NF * 32;
    uint64_t *wbar = bars + warp * NST;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(&wbar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (NF > 15 && P.nfreq < NF) {
        // generic path: rows beyond nfreq are never copied; they must read as zero
        for (int s = 0; s < NST; ++s)
            for (int r = nrows; r < 2 * NF; ++r) wring[(s * 2 * NF + r) * 32 + lane] = 0.f;
    }
    __syncthreads();
    const int count = meta[12] + meta[13];   // entries of the group that are not skipped

    const int px0 = tile * TP + warp * 32;   // first pixel of this warp
    const bool warp_has_pixels = (int64_t)px0 < npix;
    const uint32_t box_bytes = (uint32_t)nrows * 32u * 4u;
    uint64_t policy = 0;
    if (P.use_bulk) policy = P.evict_first ? policy_evict_first() : policy_evict_normal();

    auto issue = [&](int i) {   // lane 0 only
        const int s = i % NST;
        mbar_expect_tx(&wbar[s], box_bytes);
        tma_box_g2s(wring + s * 2 * NF * 32, &tmap, px0, s_drow[i], &wbar[s], policy);
    };
    if (P.use_bulk && warp_has_pixels && lane == 0)
        for (int i = 0; i < NST && i < count; ++i) issue(i);

    // row offsets (in floats) of this pixel's table rows inside an entry's table block
    const int r_fd = k0 * NROW, r_g = (cfg.K[0] + k1) * NROW, r_dg = (cfg.K[0] + cfg.K[1] + k1) * NROW,
              r_fs = (cfg.K[0] + 2 * cfg.K[1] + k2) * NROW;

    for (int i = 0; i < count; ++i) {
        const int s = i % NST;
        const float *tb = s_tab[i];
        if (live && i + 1 < count) {   // next entry's rows on their way to L1 while this entry is computed
            const float *tn = s_tab[i + 1];
            prefetch_row(tn + r_fd); prefetch_row(tn + r_g); prefetch_row(tn + r_fs);
            if (MODE == MODE_GRAD) prefetch_row(tn + r_dg);
        }
        PixelIn<NF> in;
        in.st = wring + s * 2 * NF * 32 + lane;
        if (warp_has_pixels) {
            if (P.use_bulk) {
                mbar_wait(&wbar[s], (uint32_t)((i / NST) & 1));
            } else {
                const int64_t row0 = s_drow[i];
                for (int r = 0; r < nrows; ++r)
                    wring[(s * 2 * NF + r) * 32 + lane] = (p < npix) ? P.d[(row0 + r) * npix + p] : 0.f;
                __syncwarp();
            }
        }

        float t0 = 0.f, t1 = 0.f, t2 = 0.f, t3 = 0.f;
        if (live) {
            // the pixel is its own cell: the per-cell and the per-pixel part of cs_math.cuh in one pass over the bands
            constexpr bool kGrad = (MODE == MODE_GRAD);
            const float2 *w2 = reinterpret_cast<const float2 *>(P.kc.w);
            const float2 *lnd2 = reinterpret_cast<const float2 *>(P.kc.lnd);
            const float2 *lns2 = reinterpret_cast<const float2 *>(P.kc.lns);
            const float4 *rFd = reinterpret_cast<const float4 *>(tb + r_fd), *rG = reinterpret_cast<const float4 *>(tb + r_g);
            const float4 *rdG = reinterpret_cast<const float4 *>(tb + r_dg), *rFs = reinterpret_cast<const float4 *>(tb + r_fs);
            CellSums S;
            PixSums A;
            cell_sums_zero(S);
            pix_sums_zero(A);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 vFd = __ldg(rFd + q), vG = __ldg(rG + q), vFs = __ldg(rFs + q);
                const float4 vdG = kGrad ? __ldg(rdG + q) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int j = 2 * q + h;
                    const float2 Fd = h ? make_float2(vFd.z, vFd.w) : make_float2(vFd.x, vFd.y);
                    const float2 G = h ? make_float2(vG.z, vG.w) : make_float2(vG.x, vG.y);
                    const float2 dG = h ? make_float2(vdG.z, vdG.w) : make_float2(vdG.x, vdG.y);
                    const float2 as = h ? make_float2(vFs.z, vFs.w) : make_float2(vFs.x, vFs.y);
                    const float2 wd = cell_pair<kGrad>(S, Fd, G, dG, as, w2[j], lnd2[j], lns2[j]);
                    pix_pair<kGrad>(A, wd, as, dG, w2[j], lnd2[j], lns2[j], in.dq(j), in.du(j));
                }
            }
            CellScal C;
            cell_finish<kGrad>(S, P.kc.inv_m00, C);
            if (C.bad != 0.f) atomicOr(P.err, ERR_SINGULAR);
            float sq[3], su[3], ll;
            pix_solve(A, C, P.kc.inv_m00, sq, su, ll);
            if (MODE == MODE_VALUE) {
                t3 = ll;
            } else if (MODE == MODE_CHI2) {
                const float2 *iw2 = reinterpret_cast<const float2 *>(P.kc.invw);
                ChiCoef K;
                chi_coef(sq, su, K);
                ChiSums X;
                X.q = X.u = make_float2(0.f, 0.f);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 vFd = __ldg(rFd + q), vG = __ldg(rG + q), vFs = __ldg(rFs + q);
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int j = 2 * q + h;
                        const float2 Fd = h ? make_float2(vFd.z, vFd.w) : make_float2(vFd.x, vFd.y);
                        const float2 G = h ? make_float2(vG.z, vG.w) : make_float2(vG.x, vG.y);
                        const float2 as = h ? make_float2(vFs.z, vFs.w) : make_float2(vFs.x, vFs.y);
                        const float2 wd = mul2(w2[j], mul2(Fd, G));   // as in cell_pair
                        pix_chi2_pair(X, K, wd, as, w2[j], iw2[j], in.dq(j), in.du(j));
                    }
                }
                t3 = (C.bad != 0.f) ? CUDART_INF_F : hsum(X.q) + hsum(X.u);
            } else if (MODE == MODE_GRAD) {
                pix_grad_terms(A, C, sq, su, t0, t1, t2);
                t3 = ll;
            } else if (MODE == MODE_CMBVAR) {
                t0 = sq[0]; t1 = su[0]; t2 = sq[0] * sq[0]; t3 = su[0] * su[0];
            } else {
                float *o = P.maps_out + (int64_t)(grp.start + i) * 6 * npix + p;
                o[0] = sq[0]; o[npix] = su[0]; o[2 * npix] = sq[1]; o[3 * npix] = su[1];
                o[4 * npix] = sq[2]; o[5 * npix] = su[2];
            }
        } else if (MODE == MODE_MAPS && p < npix) {
            float *o = P.maps_out + (int64_t)(grp.start + i) * 6 * npix + p;
#pragma unroll
            for (int c = 0; c < 6; ++c) o[c * npix] = 0.f;
        }
        if (warp_has_pixels && P.use_bulk) {
            __syncwarp();   // every lane is done reading stage s: refill it with the entry NST ahead
            if (lane == 0 && i + NST < count) issue(i + NST);
        }
        if (kReduce) {
            float *tm = sterm + (((i / EC) & 1) * EC + (i % EC)) * 4 * TROW;
            if (!ModeTraits<MODE>::region_only) { tm[so0] = t0; tm[so1] = t1; tm[so2] = t2; }
            tm[so3] = t3;
            if ((i % EC) == EC - 1 || i == count - 1) {
                __syncthreads();
                const int i0 = i - (i % EC), nent = (i % EC) + 1;
                reduce_terms(sterm + ((i / EC) & 1) * EC * 4 * TROW, nent, tid, meta, s_desc, s_slot, s_ent + i0, P.partial, P.PS);
            }
        }
    }
}

// ----------------------------------------------------------------------------------------------------------
// a3 second level: grad[e][j] / nll[e][r] = fixed-order (ascending tile) sum over the segments of cluster j / region r,
// which are contiguous in the partial row.
// want_grad = 0: only the region outputs.
// ----------------------------------------------------------------------------------------------------------
// Cluster outputs (short slot ranges): one thread each, slots added in ascending order.  Region outputs (one slot per
// tile): one warp each, lane l adds the slots a+l, a+l+32, ... in ascending order and the 32 lane sums are combined by a
// fixed xor-shuffle tree.  Both orders are fixed, so the result is bitwise reproducible.
// Virtual thread index v: [0, ktot) clusters, [ktot_pad + 32 r, +32) region r.  grid = (ceil(nvirt_max/256), batch).
__global__ void __launch_bounds__(256) k_merge(const double *__restrict__ partial, int64_t PS, const MapDev *__restrict__ maps,
                                               const CfgDev *__restrict__ cfgs, const int32_t *__restrict__ cfg_of,
                                               const int64_t *__restrict__ param_off, int32_t nregion, int32_t want_grad,
                                               double *__restrict__ nll, double *__restrict__ grad, const int32_t *__restrict__ skip) {
    const int e = blockIdx.y, lane = threadIdx.x & 31;
    if (skip && skip[e] != 0) return;
    const CfgDev *c = cfgs + cfg_of[e];
    const int K0 = c->K[0], K1 = c->K[1], ktot = want_grad ? c->ktot : 0;
    const int kpad = (ktot + 31) & ~31;
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    const double *erow = partial + (int64_t)e * PS;
    if (v < ktot) {
        int t, k;
        if (v < K0) { t = 0; k = v; }
        else if (v < K0 + K1) { t = 1; k = v - K0; }
        else { t = 2; k = v - K0 - K1; }
        const int32_t *ksegptr = maps[c->map[t]].ksegptr;
        const double *row = erow + c->segbase[t];
        const int a = ksegptr[k], b = ksegptr[k + 1];
        double acc = 0.0;
#pragma unroll 4
        for (int q = a; q < b; ++q) acc += row[q];
        grad[param_off[e] + v] = acc;
    } else if (v >= kpad && (v - kpad) >> 5 < nregion) {
        const int r = (v - kpad) >> 5;
        const int32_t *ksegptr = maps[c->map[3]].ksegptr;
        const double *row = erow + c->segbase[3];
        const int a = ksegptr[r], b = ksegptr[r + 1];
        double acc = 0.0;
#pragma unroll 4
        for (int q = a + lane; q < b; q += 32) acc += row[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) nll[(int64_t)e * nregion + r] = acc;
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

}  // namespace cs
