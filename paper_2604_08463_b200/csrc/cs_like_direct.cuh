// cs_like_direct.cuh -- k_like_direct: the fused per-pixel kernel (a2 + first level of a3, a4, f1) in its direct form.
//
// Every pixel is its own cell: the thread gathers the four table rows of each of its two positions and runs the
// per-cell and the per-pixel part of the arithmetic (cs_math.cuh, T = float2, lanes = the two pixels) in one pass over
// the bands.  It needs no cell plan and no private data copy, so it serves
//   - configurations that stay in place (cells too small for the sorted layout to pay, e.g. K ~ npix, the paper's own
//     optimum for beta_d, Table 2; or the context option CS_LAYOUT_INPLACE),
//   - component maps (a4), which are written in the caller's pixel order,
//   - and, forced by the context option CS_FORM_DIRECT, any configuration on whatever layout it has (tests: both
//     kernels give the same bits).
// Persistent grid and data ring as in k_like_sc (cs_pipe.cuh): warps 0-7 consume, warp 8 loads.  First level of a3:
// each thread stores its terms at the rank its positions have in the tile's (cluster, position) order; every EC
// entries the consumers meet at a named barrier and sum the segments (one thread per (entry, term, segment), fp64,
// the chunk tree of cs_math.cuh) into the partial buffer.  The term buffer is double buffered.
#pragma once
#include <type_traits>
#include "cs_pipe.cuh"
#include "cs_math.cuh"
#include "cs_tables.cuh"   // powerlaw_value: the per-pixel beta_d path evaluates the table kernel's own expression

namespace cs {

constexpr int DR_ND = 2;                 // data ring depth (deeper adds nothing, cs_like_sc.cuh; the rest of the SM's
                                         // 228 KB stays L1, which the table rows of the next entry are prefetched into)
constexpr int DR_EC = 2;                 // entries buffered between reduce phases
constexpr int DR_THREADS = NCONS + 32;   // 288
constexpr int TROW = TPX + 4;            // floats per term row: TPX ranks + a dump slot for positions without a rank

template <int NF>
struct DirectDepth { static constexpr int value = DR_ND; };

template <int NF>
constexpr size_t direct_smem_bytes() {
    return (size_t)DirectDepth<NF>::value * 2 * NF * TPX * 4   // data ring
           + (size_t)2 * DR_EC * 4 * TROW * 4                  // double-buffered terms
           + 2 * DirectDepth<NF>::value * 8                    // mbarriers
           + 2 * DR_EC * 4 + 16 * 4;                           // entry ids of the buffered terms, meta
}

// First level of the ordered reduction (a3) for `nent` buffered entries: one thread per (entry, term, segment); a
// segment is a contiguous run of the rank-ordered terms of one cluster, summed in fp64 in the fixed chunk order of
// cs_math.cuh and stored at the segment's cluster-major slot of the entry's partial row.
template <int MODE>
__device__ __forceinline__ void direct_reduce(const float *tbuf, int nent, int tid, const LikeParams &P, const CfgDev *cf, int tile,
                                              const int32_t *ents) {
    constexpr int T0 = ModeTraits<MODE>::region_only ? 3 : 0;
    int s0[4], cum[5];
    cum[0] = 0;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const MapDev *m = P.maps + ((MODE == MODE_CMBVAR) ? cf->map[3] : cf->map[t]);
        s0[t] = __ldg(m->segptr + tile);
        cum[t + 1] = cum[t] + ((t >= T0) ? __ldg(m->segptr + tile + 1) - s0[t] : 0);
    }
    const int tot = cum[4];
    for (int wi = tid; wi < nent * tot; wi += NCONS) {
        const int ent = wi / tot, r = wi - ent * tot;
        const int t = (r >= cum[1]) + (r >= cum[2]) + (r >= cum[3]);
        const int ls = r - cum[t];
        const MapDev *m = P.maps + ((MODE == MODE_CMBVAR) ? cf->map[3] : cf->map[t]);
        const uint32_t desc = __ldg(m->segdesc + s0[t] + ls);
        const int start = desc & 0x1ff, len = (int)(desc >> 9) + 1;
        const int slot = ((MODE == MODE_CMBVAR) ? t * m->nseg : cf->segbase[t]) + __ldg(m->segslot + s0[t] + ls);
        P.partial[(int64_t)ents[ent] * P.PS + slot] = segment_sum(tbuf + (ent * 4 + t) * TROW, start, len);
    }
}

template <int NF, int MODE>
__global__ void __launch_bounds__(DR_THREADS, 1) k_like_direct(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ LikeParams P) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int STAGE = 2 * NF * TPX;
    constexpr int ND = DirectDepth<NF>::value, EC = DR_EC;
    constexpr bool kGrad = ModeTraits<MODE>::grad;
    constexpr bool kReduce = ModeTraits<MODE>::reduce;
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *sterm = ring + ND * STAGE;
    uint64_t *bars = reinterpret_cast<uint64_t *>(sterm + 2 * EC * 4 * TROW);
    uint64_t *full_d = bars, *empty_d = bars + ND;
    int32_t *s_ent = reinterpret_cast<int32_t *>(bars + 2 * ND);   // [2][EC] entry ids of the buffered terms

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < ND; ++s) { mbar_init(&full_d[s], 1); mbar_init(&empty_d[s], NCONS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (NF * 2 != 2 * P.nfreq) {   // generic band count: rows beyond nfreq are never copied; they must read as zero
        for (int i = tid; i < ND * STAGE; i += DR_THREADS) ring[i] = 0.f;
    }
    __syncthreads();
    if (warp == NCONS / 32) {
        loader_loop<NF, ND>(&tmap, P, ring, full_d, empty_d, lane);
        return;
    }

    // ---------------- consumers ----------------
    const float *st0 = ring + (tid >> 7) * (2 * NF * HALF) + ((2 * tid) & (HALF - 1));
    const KConst &kc = P.kc;
    Walk w;
    walk_init(w, P);
    int n = 0;        // live entries so far
    int nbuf = 0;     // entries in the current term buffer
    int blk = 0;      // reduce blocks so far (buffer = blk & 1)
    while (walk_next(w, P)) {
        const CfgDev *cf = P.cfgs + w.run.cfg;
        const int32_t *mp = P.ring_maps ? cf->rmap : cf->map;
        const int64_t posA = (int64_t)w.tile * TPX + 2 * tid;
        const int64_t npos = (cf->sorted && !P.ring_maps) ? (int64_t)cf->ntile * TPX : P.npix;
        const bool inA = posA < npos, inB = posA + 1 < npos;
        int k0A = -1, k1A = -1, k2A = -1, k0B = -1, k1B = -1, k2B = -1;
        if (inA) { k0A = __ldg(P.maps[mp[0]].idx + posA); k1A = __ldg(P.maps[mp[1]].idx + posA); k2A = __ldg(P.maps[mp[2]].idx + posA); }
        if (inB) { k0B = __ldg(P.maps[mp[0]].idx + posA + 1); k1B = __ldg(P.maps[mp[1]].idx + posA + 1); k2B = __ldg(P.maps[mp[2]].idx + posA + 1); }
        const bool liveA = (k0A >= 0) && (k1A >= 0) && (k2A >= 0), liveB = (k0B >= 0) && (k1B >= 0) && (k2B >= 0);
        // float offset of each position's slot in each term row: its rank in the tile's (cluster, position) order of the
        // reducing map, or the dump slot TPX when the position has no cluster there
        int soA[4] = {TPX, TROW + TPX, 2 * TROW + TPX, 3 * TROW + TPX}, soB[4] = {TPX, TROW + TPX, 2 * TROW + TPX, 3 * TROW + TPX};
        if (kReduce) {
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                if (ModeTraits<MODE>::region_only && t < 3) continue;
                const MapDev *m = P.maps + ((MODE == MODE_CMBVAR) ? mp[3] : mp[t]);
                // a position masked in another map still owns a rank here: its slot must read 0
                if (inA) { const int r = __ldg(m->rank + posA); if (r != NORANK) soA[t] = t * TROW + r; }
                if (inB) { const int r = __ldg(m->rank + posA + 1); if (r != NORANK) soB[t] = t * TROW + r; }
            }
        }
        // row offsets (in floats) of the positions' table rows inside an entry's table block (row 0 for dead positions)
        const int K0 = cf->K[0], K1 = cf->K[1];
        const int rA_fd = max(k0A, 0) * NROW, rA_g = (K0 + max(k1A, 0)) * NROW, rA_dg = (K0 + K1 + max(k1A, 0)) * NROW,
                  rA_fs = (K0 + 2 * K1 + max(k2A, 0)) * NROW;
        const int rB_fd = max(k0B, 0) * NROW, rB_g = (K0 + max(k1B, 0)) * NROW, rB_dg = (K0 + K1 + max(k1B, 0)) * NROW,
                  rB_fs = (K0 + 2 * K1 + max(k2B, 0)) * NROW;

        // beta_d (nearly) per pixel (CfgDev::pixbeta): every beta_d row would be built, written and read for one or two
        // pixels, 128 B of traffic per pixel-eval next to the 120 B of data; the row's values are evaluated here instead,
        // from the parameter copy, in compensated fp32 for both pixels at once (cs_tables.cuh: powerlaw_pair_f32)
        // The entry loop exists twice, with and without that path, so that the ordinary one keeps its registers and
        // schedule (with the branch inside one loop the component maps ran a quarter slower).
        auto entry_loop = [&](auto pb) {
        constexpr bool pixbeta = decltype(pb)::value;
        for (int k = w.k; k < w.kend; ++k) {
            const int e = __ldg(P.elist + w.run.estart + k);
            if (P.skip && __ldg(P.skip + e) != 0) continue;
            const int sd = n % ND;
            const float *tb = P.tab + __ldg(&P.pinfo[w.run.estart + k].tab_row) * NROW;
            const float *st = st0 + sd * STAGE;
            float2 bh = make_float2(0.f, 0.f), bl = bh;   // beta_d of the two pixels as float pairs
            if (pixbeta) {
                const double *pe = P.pcopy + __ldg(&P.pinfo[w.run.estart + k].param_off);
                const double betaA = __ldg(pe + max(k0A, 0)), betaB = __ldg(pe + max(k0B, 0));
                bh = make_float2((float)betaA, (float)betaB);
                bl = make_float2((float)(betaA - (double)bh.x), (float)(betaB - (double)bh.y));
            }
            if (k + 1 < w.kend) {   // the next entry's rows on their way to L1 while this entry is computed
                const float *tn = P.tab + __ldg(&P.pinfo[w.run.estart + k + 1].tab_row) * NROW;
                if (liveA) { if (!pixbeta) prefetch_row(tn + rA_fd); prefetch_row(tn + rA_g); prefetch_row(tn + rA_fs); if (kGrad) prefetch_row(tn + rA_dg); }
                if (liveB) { if (!pixbeta) prefetch_row(tn + rB_fd); prefetch_row(tn + rB_g); prefetch_row(tn + rB_fs); if (kGrad) prefetch_row(tn + rB_dg); }
            }
            mbar_wait(&full_d[sd], (uint32_t)((n / ND) & 1));
            const float4 *aFd = reinterpret_cast<const float4 *>(tb + rA_fd), *aG = reinterpret_cast<const float4 *>(tb + rA_g);
            const float4 *adG = reinterpret_cast<const float4 *>(tb + rA_dg), *aFs = reinterpret_cast<const float4 *>(tb + rA_fs);
            const float4 *bFd = reinterpret_cast<const float4 *>(tb + rB_fd), *bG = reinterpret_cast<const float4 *>(tb + rB_g);
            const float4 *bdG = reinterpret_cast<const float4 *>(tb + rB_dg), *bFs = reinterpret_cast<const float4 *>(tb + rB_fs);
            CellSums<float2> S;
            PixSums A;
            cell_sums_zero(S);
            pix_sums_zero(A);
            float2 wdk[NROW], wsk[NROW];   // kept for the second pass of MODE_CHI2 only
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float4 xFd, yFd;
                if (pixbeta) {
                    float a[4], b[4];
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const int f = 4 * q + h;   // bands beyond nfreq: cdf = 0
                        const float2 v = powerlaw_pair_f32(P.cdf[f], P.l2h[f], P.l2l[f], bh, bl);
                        a[h] = v.x; b[h] = v.y;
                    }
                    xFd = make_float4(a[0], a[1], a[2], a[3]); yFd = make_float4(b[0], b[1], b[2], b[3]);
                } else {
                    xFd = __ldg(aFd + q); yFd = __ldg(bFd + q);
                }
                const float4 xG = __ldg(aG + q), xFs = __ldg(aFs + q);
                const float4 yG = __ldg(bG + q), yFs = __ldg(bFs + q);
                float4 xdG = make_float4(0.f, 0.f, 0.f, 0.f), ydG = xdG;
                if (kGrad) { xdG = __ldg(adG + q); ydG = __ldg(bdG + q); }
                const float2 vFd[4] = {{xFd.x, yFd.x}, {xFd.y, yFd.y}, {xFd.z, yFd.z}, {xFd.w, yFd.w}};
                const float2 vG[4] = {{xG.x, yG.x}, {xG.y, yG.y}, {xG.z, yG.z}, {xG.w, yG.w}};
                const float2 vdG[4] = {{xdG.x, ydG.x}, {xdG.y, ydG.y}, {xdG.z, ydG.z}, {xdG.w, ydG.w}};
                const float2 vFs[4] = {{xFs.x, yFs.x}, {xFs.y, yFs.y}, {xFs.z, yFs.z}, {xFs.w, yFs.w}};
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int f = 4 * q + h;
                    if (f < NF) {
                        const float2 dq = *reinterpret_cast<const float2 *>(st + (2 * f) * HALF);
                        const float2 du = *reinterpret_cast<const float2 *>(st + (2 * f + 1) * HALF);
                        CellCols<float2> C;
                        cell_band<kGrad>(S, C, vFd[h], vG[h], vdG[h], vFs[h], kc.w[f], kc.lnd[f], kc.lns[f]);
                        pix_band<kGrad>(A, C, kc.w[f], dq, du);
                        if (MODE == MODE_CHI2) { wdk[f] = C.wd; wsk[f] = C.ws; }
                    }
                }
            }
            CellScal<float2> C;
            cell_finish<kGrad>(S, kc.inv_m00, C);
            if ((liveA && C.bad.x != 0.f) || (liveB && C.bad.y != 0.f)) atomicOr(P.err, ERR_SINGULAR);
            float2 sq[3], su[3], ll;
            pix_solve(A, C, kc.inv_m00, sq, su, ll);
            float2 t0 = make_float2(0.f, 0.f), t1 = t0, t2 = t0, t3 = t0;
            if (MODE == MODE_CHI2) {
                float2 xq = make_float2(0.f, 0.f), xu = xq;
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    const float2 dq = *reinterpret_cast<const float2 *>(st + (2 * f) * HALF);
                    const float2 du = *reinterpret_cast<const float2 *>(st + (2 * f + 1) * HALF);
                    pix_chi2_band(xq, xu, sq, su, wdk[f], wsk[f], kc.w[f], kc.invw[f], dq, du);
                }
                t3 = sel_inf(C.bad, add_(xq, xu));
            }
            __syncwarp();   // every lane is done reading the stage
            if (lane == 0) mbar_arrive(&empty_d[sd]);
            if (MODE == MODE_VALUE) {
                t3 = ll;
            } else if (MODE == MODE_GRAD) {
                pix_grad_terms(A, C, sq, su, t0, t1, t2);
                t3 = ll;
            } else if (MODE == MODE_CMBVAR) {
                t0 = sq[0]; t1 = su[0]; t2 = mul_(sq[0], sq[0]); t3 = mul_(su[0], su[0]);
            } else if (MODE == MODE_MAPS) {
                float *o = P.maps_out + (int64_t)(w.run.estart + k) * P.maps_planes * P.npix + posA;
                const float2 v[6] = {sq[0], su[0], sq[1], su[1], sq[2], su[2]};
                const bool vec = inB && ((P.npix & 1) == 0) && ((reinterpret_cast<uintptr_t>(P.maps_out) & 7) == 0);
#pragma unroll
                for (int c = 0; c < 6; ++c) {
                    if (c >= P.maps_planes) break;
                    const float a = liveA ? v[c].x : 0.f, b = liveB ? v[c].y : 0.f;
                    if (vec) {
                        *reinterpret_cast<float2 *>(o + c * P.npix) = make_float2(a, b);
                    } else {
                        if (inA) o[c * P.npix] = a;
                        if (inB) o[c * P.npix + 1] = b;
                    }
                }
            }
            if (kReduce) {
                float *tm = sterm + ((blk & 1) * EC + nbuf) * 4 * TROW;
                if (!ModeTraits<MODE>::region_only) {
                    tm[soA[0]] = liveA ? t0.x : 0.f; tm[soB[0]] = liveB ? t0.y : 0.f;
                    tm[soA[1]] = liveA ? t1.x : 0.f; tm[soB[1]] = liveB ? t1.y : 0.f;
                    tm[soA[2]] = liveA ? t2.x : 0.f; tm[soB[2]] = liveB ? t2.y : 0.f;
                }
                tm[soA[3]] = liveA ? t3.x : 0.f; tm[soB[3]] = liveB ? t3.y : 0.f;
                if (tid == 0) s_ent[(blk & 1) * EC + nbuf] = e;
                if (++nbuf == EC) {
                    __threadfence_block();
                    named_sync(1, NCONS);
                    direct_reduce<MODE>(sterm + (blk & 1) * EC * 4 * TROW, nbuf, tid, P, cf, w.tile, s_ent + (blk & 1) * EC);
                    nbuf = 0; ++blk;
                }
            }
            ++n;
        }
        };
        if (cf->pixbeta != 0) entry_loop(std::true_type{}); else entry_loop(std::false_type{});
        if (kReduce && nbuf > 0) {   // the tile changes (or the share ends): flush what is buffered with this tile's plan
            __threadfence_block();
            named_sync(1, NCONS);
            direct_reduce<MODE>(sterm + (blk & 1) * EC * 4 * TROW, nbuf, tid, P, cf, w.tile, s_ent + (blk & 1) * EC);
            nbuf = 0; ++blk;
        }
    }
}

}  // namespace cs
