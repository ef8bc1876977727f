// cs_like_sc.cuh -- k_like_sc: the fused per-pixel kernel (a2 + first level of a3, f1) on the sorted layout.
//
// Everything in Eq. 5/6/17 that depends on the parameters depends on the pixel only through its cluster triple
// (k0,k1,k2): the weighted columns N^-1 a_d, N^-1 a_s and their derivatives, the matrix M = A^T N^-1 A,
// its LDL^T factors and the nine contractions P_{theta,c} = sum_f w_f (da_f/dtheta) A_{f,c}.  Pixels with the same
// triple (and region) form a *cell*.  In the sorted layout (cs_internal.h) the pixels of a cell are consecutive and every
// consumer thread owns two positions of one cell, so per entry a builder lane evaluates the per-cell part once per cell
// of the tile, and a pixel-eval is left with
//
//     b_S  = A^T N^-1 d_S                        (3 dots per Stokes)            Eq. 5
//     c_S  = (dA/dtheta)^T N^-1 d_S              (3 dots per Stokes)
//     s_S  = M^-1 b_S  via the cell's LDL^T ;   ll = -1/2 sum_S b_S . s_S       Eq. 5, 6
//     g_th = - sum_S s_{S,c(th)} ( c_{S,th} - sum_c P_{th,c} s_{S,c} )          Eq. 17 with r = d - A s expanded
//
// evaluated for the thread's two pixels at once: 12 packed FFMA2 per band whose coefficient operand is a per-cell
// scalar (broadcast operand form), data read as one LDS.64 per band and Stokes parameter.
//
// Persistent grid: one CTA per SM, each walking a contiguous, equal share of all (tile, entry) units (cs_pipe.cuh).
// CTA = 14 warps (128 registers per thread), warp-specialised; every hand-over is an mbarrier full/empty pair or a hardware named barrier, no
// CTA-wide barrier after the prologue:
//   warps 0-7    consumers: positions (2t, 2t+1) of the 512-position tile per thread, one entry after the other
//   warps 8-9    reducers : first level of the ordered fp64 reduction (a3) of the pair sums the consumers leave behind;
//                           warp r owns term-ring slot r and the entries n = r (mod 2)
//   warps 10-12  builders : lane c builds the cells c and c + 32 of the tile (five weighted columns, LDL^T, P); warp b
//                           owns cell-table slot b and the entries n = b (mod 3).  Three of them, and each prefetches the
//                           rows of its next entry to L1, because under a saturated HBM stream the L2 round trip of a
//                           cell's four table rows takes about as long as a whole entry
//   warp  13     loader   : one 60-KB bulk copy per entry into the data ring (two stages: measured, a deeper ring
//                           adds nothing once the consumers release a stage as soon as it is read), and one bulk copy
//                           per tile of the tile's header (cs_internal.h) into the header ring, one tile ahead: what the
//                           other roles need to know about a tile (cell of every thread, ranks, cell rows, reducer plan)
//                           is in shared memory before they get there, so a change of tile costs no dependent global
//                           load -- a clustering scan (config 3) changes tile and configuration with every entry
// shared memory: data ring [ND][2 halves][2*NF][256] | cell tables [NC][CELL_CAP][CROW] | term ring [NT][4][256] fp64 |
//                header ring [NH][HDR_CAP_WORDS] | barriers
#pragma once
#include "cs_pipe.cuh"
#include "cs_math.cuh"

namespace cs {

#ifndef CS_SC_ND
#define CS_SC_ND 2
#endif
#ifndef CS_SC_NBW
#define CS_SC_NBW 3
#endif
constexpr int SC_ND = CS_SC_ND; // data ring depth 
template <int NF>
struct ScDepth { static constexpr int value = SC_ND; };
constexpr int SC_NC = CS_SC_NBW; // cell-table ring depth = builder warps
constexpr int SC_NBW = CS_SC_NBW; // builder warps (warp b takes the entries n = b mod SC_NBW; SC_NC is a multiple of it)
constexpr int SC_NT = 2;        // term ring depth = reducer warps
constexpr int SC_THREADS = NCONS + (SC_NT + SC_NBW + 1) * 32;   // 448
constexpr int SC_WARP_RED = NCONS / 32, SC_WARP_BUILD = SC_WARP_RED + SC_NT, SC_WARP_LOAD = SC_WARP_BUILD + SC_NBW;
constexpr int SC_NH = 4;        // header ring depth: the header of tile i+1 is fetched while tile i is worked on, into the
                                // slot tile i-3 used, which every role has left by then
constexpr int SC_HDR_USERS = NCONS / 32 + SC_NBW + SC_NT;   // warps that read a header and hand its slot back

template <int NF>
constexpr size_t sc_smem_bytes() {
    return (size_t)ScDepth<NF>::value * 2 * NF * TPX * 4   // data ring
           + (size_t)SC_NC * CELL_CAP * CROW * 4       // cell tables
           + (size_t)SC_NT * 4 * NCONS * 8             // term ring (fp64 pair sums)
           + (size_t)SC_NH * HDR_CAP_WORDS * 4         // header ring
           + (2 * ScDepth<NF>::value + 2 * SC_NC + SC_NT + 2 * SC_NH) * 8   // mbarriers
           + 16;
}

// Reducer plan of a tile (part of its header): every (term, cluster) segment of <= SEG_MAX rank-ordered terms is cut
// into 1..4 chunks of <= CHUNK_LEN ranks.  In the sorted layout all starts and lengths are even; the plan is kept in pairs:
// cdesc[chunk] = first pair (8 bits) | (pairs-1) << 8 | term << 10;
// sdesc[segment] = first pair (8 bits) | (chunks-1) << 8 | term << 10; slot[segment] = slot in the entry's partial row.
// Modes that reduce only the region term use the part of the plan that belongs to term 3; MODE_CMBVAR reduces four
// terms that all follow the region map: term 3's part with the term replaced and the slots re-based.
//
// First level of the ordered reduction (a3) of one entry by a reducer warp, in fp64 and in a fixed order:
// step 1, one lane per chunk: (y0 + y1) + (y2 + y3) over the chunk's <= 4 pair sums (cs_math.cuh: chunk_tree), left in
// place of the chunk's first pair sum; step 2, one lane per segment: the segment's chunk sums left to right, stored at
// the segment's cluster-major slot of the entry's partial row.  Two chunks / segments per lane and round are in flight.
__device__ __forceinline__ double sc_chunk(const double *tbuf, uint32_t d, int &at) {
    const int p0 = d & 0xff, np = (int)((d >> 8) & 3) + 1, t = (int)(d >> 10);
    at = t * NCONS + p0;
    const double *y = tbuf + at;
    const double y0 = y[0], y1 = np > 1 ? y[1] : 0.0, y2 = np > 2 ? y[2] : 0.0, y3 = np > 3 ? y[3] : 0.0;
    return chunk_tree(y0, y1, y2, y3);
}
__device__ __forceinline__ double sc_segment(const double *tbuf, uint32_t d) {
    const int p0 = d & 0xff, cnt = (int)((d >> 8) & 3) + 1, t = (int)(d >> 10);
    const double *y = tbuf + t * NCONS + p0;
    double acc = y[0];
    if (cnt > 1) acc += y[CHUNK_LEN / 2];
    if (cnt > 2) acc += y[CHUNK_LEN];
    if (cnt > 3) acc += y[3 * CHUNK_LEN / 2];
    return acc;
}
template <int MODE>
__device__ __forceinline__ void sc_reduce_entry(double *tbuf, int lane, const uint32_t *h, double *__restrict__ prow) {
    constexpr bool kTerm3 = ModeTraits<MODE>::region_only || MODE == MODE_CMBVAR;
    constexpr bool kRep = MODE == MODE_CMBVAR;
    const uint16_t *cdesc = reinterpret_cast<const uint16_t *>(h + h[HM_OFF_CDESC]);
    const uint16_t *sdesc = reinterpret_cast<const uint16_t *>(h + h[HM_OFF_SDESC]);
    const int32_t *slot = reinterpret_cast<const int32_t *>(h + h[HM_OFF_SLOT]);
    const int c_lo = kTerm3 ? (int)h[HM_CBASE3] : 0, s_lo = kTerm3 ? (int)h[HM_SBASE3] : 0;
    const int ncr = (int)h[HM_NCHUNK] - c_lo, nsr = (int)h[HM_NSEG] - s_lo;
    const int nsegreg = (int)h[HM_NSEGREG], segbase3 = (int)h[HM_SEGBASE3];
    auto chunk_desc = [&](int r) -> uint32_t {
        if (!kRep) return cdesc[c_lo + r];
        const int rep = r / ncr;
        return (uint32_t)(cdesc[c_lo + r - rep * ncr] & 0x3ff) | ((uint32_t)rep << 10);
    };
    auto seg_desc = [&](int r, int &sl) -> uint32_t {
        if (!kRep) { sl = slot[s_lo + r]; return sdesc[s_lo + r]; }
        const int rep = r / nsr, i = r - rep * nsr;
        sl = rep * nsegreg + (slot[s_lo + i] - segbase3);
        return (uint32_t)(sdesc[s_lo + i] & 0x3ff) | ((uint32_t)rep << 10);
    };
    const int nchunk = (kRep ? 4 : 1) * ncr, nseg = (kRep ? 4 : 1) * nsr;
    for (int r = lane; r < nchunk; r += 64) {
        int a0, a1 = 0;
        const bool two = r + 32 < nchunk;
        const uint32_t d0 = chunk_desc(r), d1 = two ? chunk_desc(r + 32) : 0u;
        const double c0 = sc_chunk(tbuf, d0, a0);
        double c1 = 0.0;
        if (two) c1 = sc_chunk(tbuf, d1, a1);
        tbuf[a0] = c0;
        if (two) tbuf[a1] = c1;
    }
    __syncwarp();
    for (int r = lane; r < nseg; r += 64) {
        const bool two = r + 32 < nseg;
        int slot0 = 0, slot1 = 0;
        const uint32_t d0 = seg_desc(r, slot0), d1 = two ? seg_desc(r + 32, slot1) : 0u;
        const double v0 = sc_segment(tbuf, d0);
        double v1 = 0.0;
        if (two) v1 = sc_segment(tbuf, d1);
        prow[slot0] = v0;
        if (two) prow[slot1] = v1;
    }
    __syncwarp();
}

// Loader of the sorted-cell kernel (one lane): walks the CTA's pieces (a tile and a range of entries of one run); for
// piece i it first sends off the header of piece i+1, then asks for the header range of piece i+2 (a load whose result
// is not needed before the next round), then streams the entries of piece i into the data ring.
template <int NF, int ND>
__device__ __forceinline__ void sc_loader(const LikeParams &P, float *ring, uint32_t *hdr, uint64_t *full_d, uint64_t *empty_d,
                                          uint64_t *full_h, uint64_t *empty_h) {
    constexpr int STAGE = 2 * NF * TPX;   // floats per stage
    const int nrows = 2 * P.nfreq;
    const uint64_t policy = P.evict_first ? policy_evict_first() : policy_evict_normal();
    const uint64_t keep = policy_evict_normal();
    auto hdr_range = [](const Walk &x) { return make_int2(__ldg(x.run.hdrptr + x.tile), __ldg(x.run.hdrptr + x.tile + 1)); };
    auto send_header = [&](int ip, const Walk &x, int2 hr) {
        const int s = ip % SC_NH;
        mbar_wait(&empty_h[s], (uint32_t)(((ip / SC_NH) & 1) ^ 1));
        const uint32_t bytes = (uint32_t)(hr.y - hr.x) * 16u;
        mbar_expect_tx(&full_h[s], bytes);
        bulk_g2s(hdr + s * HDR_CAP_WORDS, x.run.hdr + (int64_t)hr.x * 4, bytes, &full_h[s], keep);
    };
    Walk w0, w1, w2;   // pieces i, i+1, i+2
    walk_init(w0, P);
    if (!walk_next(w0, P)) return;
    w1 = w0;
    bool ok1 = walk_next(w1, P);
    int2 h1 = make_int2(0, 0);
    send_header(0, w0, hdr_range(w0));
    if (ok1) h1 = hdr_range(w1);
    int n = 0;   // live entries so far
    for (int ip = 0;; ++ip) {
        bool ok2 = false;
        int2 h2 = make_int2(0, 0);
        if (ok1) {
            send_header(ip + 1, w1, h1);
            w2 = w1;
            ok2 = walk_next(w2, P);
            if (ok2) h2 = hdr_range(w2);
        }
        for (int k = w0.k; k < w0.kend; ++k) {
            const int64_t srcinfo = __ldg(&P.pinfo[w0.run.estart + k].src);
            if (P.skip && __ldg(P.skip + __ldg(P.elist + w0.run.estart + k)) != 0) continue;
            const int s = n % ND;
            float *dst = ring + s * STAGE;
            mbar_wait(&empty_d[s], (uint32_t)(((n / ND) & 1) ^ 1));
            const uint32_t bytes = (uint32_t)nrows * TPX * 4u;
            mbar_expect_tx(&full_d[s], bytes);
            const float *src = P.dcopy + srcinfo + (int64_t)w0.tile * w0.run.tstride;
            if (NF * 2 == nrows) {
                bulk_g2s(dst, src, bytes, &full_d[s], policy);
            } else {   // generic band count: the stage keeps 2*NF rows per half, the copy only 2*nfreq
                bulk_g2s(dst, src, bytes / 2, &full_d[s], policy);
                bulk_g2s(dst + NF * 2 * HALF, src + nrows * HALF, bytes / 2, &full_d[s], policy);
            }
            ++n;
        }
        if (!ok1) break;
        w0 = w1; w1 = w2; ok1 = ok2; h1 = h2;
    }
}

// One cell (Eq. 2 columns -> five weighted columns, M, LDL^T, P; cs_math.cuh) from the entry's four table rows.
// Cell row (CROW = 68 floats): [0,16) w a_d | [16,32) w da_d/dT_d (gradient modes only) | [32,48) w a_s |
// [48,64) l10 l20 l21 1/d1 | 1/d2 P10 P11 P12 | P20 P21 P22 P30 | P31 P32 bad - | [64,68) pad.
// The beta derivatives are not stored: w da_d/dbeta_d = lnd w a_d and w da_s/dbeta_s = lns w a_s.
template <int NF, bool GRAD>
__device__ __forceinline__ void sc_build_cell(const float4 (&Fd)[4], const float4 (&G)[4], const float4 (&dG)[4], const float4 (&Fs)[4],
                                              const KConst &kc, float *__restrict__ out, int32_t *err) {
    CellSums<float> S;
    cell_sums_zero(S);
    float4 *o4 = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float vFd[4] = {Fd[q].x, Fd[q].y, Fd[q].z, Fd[q].w}, vG[4] = {G[q].x, G[q].y, G[q].z, G[q].w};
        const float vdG[4] = {dG[q].x, dG[q].y, dG[q].z, dG[q].w}, vFs[4] = {Fs[q].x, Fs[q].y, Fs[q].z, Fs[q].w};
        float wd[4] = {0.f, 0.f, 0.f, 0.f}, u1[4] = {0.f, 0.f, 0.f, 0.f}, u2[4] = {0.f, 0.f, 0.f, 0.f}, ws[4] = {0.f, 0.f, 0.f, 0.f},
              u3[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const int f = 4 * q + h;
            if (f < NF) {   // bands beyond nfreq carry w = 0 and zero table entries: their columns come out as zero
                CellCols<float> C;
                cell_band<GRAD>(S, C, vFd[h], vG[h], vdG[h], vFs[h], kc.w[f], kc.lnd[f], kc.lns[f]);
                wd[h] = C.wd; u1[h] = C.u1; u2[h] = C.u2; ws[h] = C.ws; u3[h] = C.u3;
            }
        }
        o4[q] = make_float4(wd[0], wd[1], wd[2], wd[3]);
        o4[CR_WS + q] = make_float4(ws[0], ws[1], ws[2], ws[3]);
        if (GRAD) o4[4 + q] = make_float4(u2[0], u2[1], u2[2], u2[3]);   // the other two derivative columns are one multiply
                                                                         // by a band constant away from w a_d and w a_s
    }
    CellScal<float> C;
    cell_finish<GRAD>(S, kc.inv_m00, C);
    if (C.bad != 0.f) atomicOr(err, ERR_SINGULAR);
    o4[CR_SC] = make_float4(C.l10, C.l20, C.l21, C.id1);
    o4[CR_SC + 1] = make_float4(C.id2, C.P10, C.P11, C.P12);
    o4[CR_SC + 2] = make_float4(C.P20, C.P21, C.P22, C.P30);
    o4[CR_SC + 3] = make_float4(C.P31, C.P32, C.bad, 0.f);
}

template <int NF, int MODE>
__global__ void __launch_bounds__(SC_THREADS, 1) k_like_sc(const LikeParams P) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int STAGE = 2 * NF * TPX;   // floats per data stage
    constexpr int ND = ScDepth<NF>::value, NC = SC_NC, NT = SC_NT;
    constexpr bool kGrad = ModeTraits<MODE>::grad;
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *cells = ring + ND * STAGE;
    double *sterm = reinterpret_cast<double *>(cells + NC * CELL_CAP * CROW);
    uint32_t *hdr = reinterpret_cast<uint32_t *>(sterm + NT * 4 * NCONS);
    uint64_t *bars = reinterpret_cast<uint64_t *>(hdr + SC_NH * HDR_CAP_WORDS);
    uint64_t *full_d = bars, *empty_d = bars + ND, *full_c = bars + 2 * ND, *empty_c = bars + 2 * ND + NC;
    uint64_t *empty_t = bars + 2 * ND + 2 * NC;
    uint64_t *full_h = empty_t + NT, *empty_h = full_h + SC_NH;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // ---------------- prologue (all threads) ----------------
    if (tid == 0) {
        for (int s = 0; s < ND; ++s) { mbar_init(&full_d[s], 1); mbar_init(&empty_d[s], NCONS / 32); }
        for (int s = 0; s < NC; ++s) { mbar_init(&full_c[s], 1); mbar_init(&empty_c[s], NCONS / 32); }
        for (int s = 0; s < NT; ++s) mbar_init(&empty_t[s], 1);
        for (int s = 0; s < SC_NH; ++s) { mbar_init(&full_h[s], 1); mbar_init(&empty_h[s], SC_HDR_USERS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (NF * 2 != 2 * P.nfreq) {   // generic band count: rows beyond nfreq are never copied; they must read as zero
        for (int i = tid; i < ND * STAGE; i += SC_THREADS) ring[i] = 0.f;
    }
    __syncthreads();

    if (warp == SC_WARP_LOAD) {
        if (lane == 0) sc_loader<NF, ND>(P, ring, hdr, full_d, empty_d, full_h, empty_h);
        return;
    }
    Walk w;
    walk_init(w, P);
    int n = 0;    // live entries so far (ring slots and barrier phases follow it)
    int ip = 0;   // pieces so far (header ring slot and phase)

    if (warp >= SC_WARP_BUILD) {
        // ---------------- builder warps: lane c builds the cells c and c + 32 of the current tile; warp b takes the
        // entries n = b (mod SC_NBW)
        static_assert(CELL_CAP == 64, "two cells per builder lane");
        const int mine = warp - SC_WARP_BUILD;
        for (; walk_next(w, P); ++ip) {
            const uint32_t *hd = hdr + (ip % SC_NH) * HDR_CAP_WORDS;
            mbar_wait(&full_h[ip % SC_NH], (uint32_t)((ip / SC_NH) & 1));
            const int ncell = (int)hd[HM_NCELL];
            const int4 *hrows = reinterpret_cast<const int4 *>(hd + HDR_META + HDR_CONS);
            const int4 rows0 = (lane < ncell) ? hrows[lane] : make_int4(0, 0, 0, 0);
            const int4 rows1 = (lane + 32 < ncell) ? hrows[lane + 32] : make_int4(0, 0, 0, 0);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_h[ip % SC_NH]);
            for (int k = w.k; k < w.kend; ++k) {
                const int64_t tab_row = __ldg(&P.pinfo[w.run.estart + k].tab_row);
                if (P.skip && __ldg(P.skip + __ldg(P.elist + w.run.estart + k)) != 0) continue;
                const int s = n % NC;
                if (SC_NBW > 1 && n % SC_NBW != mine) { ++n; continue; }
                const float *tb = P.tab + tab_row * NROW;
                const int nh = ncell > 32 ? 2 : 1;   // warp-uniform: most tiles hold fewer than 32 cells
                if (k + SC_NBW < w.kend) {   // this warp's next entry: its rows on their way to L1
                    const float *tn = P.tab + __ldg(&P.pinfo[w.run.estart + k + SC_NBW].tab_row) * NROW;
                    if (lane < ncell) {
                        prefetch_row(tn + (int64_t)rows0.x * NROW); prefetch_row(tn + (int64_t)rows0.y * NROW);
                        prefetch_row(tn + (int64_t)rows0.w * NROW);
                        if (kGrad) prefetch_row(tn + (int64_t)rows0.z * NROW);
                    }
                    if (lane + 32 < ncell) {
                        prefetch_row(tn + (int64_t)rows1.x * NROW); prefetch_row(tn + (int64_t)rows1.y * NROW);
                        prefetch_row(tn + (int64_t)rows1.w * NROW);
                        if (kGrad) prefetch_row(tn + (int64_t)rows1.z * NROW);
                    }
                }
#pragma unroll 1
                for (int h = 0; h < nh; ++h) {
                    const int4 rows = h ? rows1 : rows0;
                    const int c = lane + 32 * h;
                    float4 Fd[4], G[4], dG[4], Fs[4];
                    if (c < ncell) {
                        const float4 *rFd = reinterpret_cast<const float4 *>(tb + (int64_t)rows.x * NROW);
                        const float4 *rG = reinterpret_cast<const float4 *>(tb + (int64_t)rows.y * NROW);
                        const float4 *rdG = reinterpret_cast<const float4 *>(tb + (int64_t)rows.z * NROW);
                        const float4 *rFs = reinterpret_cast<const float4 *>(tb + (int64_t)rows.w * NROW);
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            Fd[q] = __ldg(rFd + q); G[q] = __ldg(rG + q); Fs[q] = __ldg(rFs + q);
                            dG[q] = kGrad ? __ldg(rdG + q) : make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                    }
                    if (h == 0) mbar_wait(&empty_c[s], (uint32_t)(((n / NC) & 1) ^ 1));
                    if (c < ncell) sc_build_cell<NF, kGrad>(Fd, G, dG, Fs, P.kc, cells + (s * CELL_CAP + c) * CROW, P.err);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&full_c[s]);
                ++n;
            }
        }
        return;
    }
    if (warp >= SC_WARP_RED) {
        // ---------------- reducer warps: first level of a3; warp r takes the entries n = r (mod NT) ----------------
        const int mine = warp - SC_WARP_RED;
        for (; walk_next(w, P); ++ip) {
            const uint32_t *h = hdr + (ip % SC_NH) * HDR_CAP_WORDS;   // the tile's plan is used in place
            mbar_wait(&full_h[ip % SC_NH], (uint32_t)((ip / SC_NH) & 1));
            for (int k = w.k; k < w.kend; ++k) {
                const int e = __ldg(P.elist + w.run.estart + k);
                if (P.skip && __ldg(P.skip + e) != 0) continue;
                const int s = n % NT;
                if (s != mine) { ++n; continue; }
                named_sync(1 + s, NCONS + 32);
                sc_reduce_entry<MODE>(sterm + s * 4 * NCONS, lane, h, P.partial + (int64_t)e * P.PS);
                if (lane == 0) mbar_arrive(&empty_t[s]);
                ++n;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_h[ip % SC_NH]);
        }
        return;
    }

    // ---------------- consumers ----------------
    const float *st0 = ring + (tid >> 7) * (2 * NF * HALF) + ((2 * tid) & (HALF - 1));
    const KConst &kc = P.kc;
    for (; walk_next(w, P); ++ip) {
        // this thread's cell and the slots of its pair sums in the four term rows (half the rank of its first position)
        mbar_wait(&full_h[ip % SC_NH], (uint32_t)((ip / SC_NH) & 1));
        const uint2 ci = reinterpret_cast<const uint2 *>(hdr + (ip % SC_NH) * HDR_CAP_WORDS + HDR_META)[tid];
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_h[ip % SC_NH]);
        const int cell = (int)(ci.x & 0xff);
        int so0, so1, so2, so3;
        if (MODE == MODE_CMBVAR) {
            so0 = (int)ci.y; so1 = NCONS + (int)ci.y; so2 = 2 * NCONS + (int)ci.y; so3 = 3 * NCONS + (int)ci.y;
        } else {
            so0 = (int)((ci.x >> 8) & 0xff); so1 = NCONS + (int)((ci.x >> 16) & 0xff); so2 = 2 * NCONS + (int)(ci.x >> 24);
            so3 = 3 * NCONS + (int)ci.y;
        }
        for (int k = w.k; k < w.kend; ++k) {
            const int e = __ldg(P.elist + w.run.estart + k);
            if (P.skip && __ldg(P.skip + e) != 0) continue;
            const int sd = n % ND, sc = n % NC, stt = n % NT;
            const float4 *crow = reinterpret_cast<const float4 *>(cells + (sc * CELL_CAP + cell) * CROW);
            const float *st = st0 + sd * STAGE;
            mbar_wait(&full_c[sc], (uint32_t)((n / NC) & 1));
            mbar_wait(&full_d[sd], (uint32_t)((n / ND) & 1));
            PixSums A;
            pix_sums_zero(A);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 WD = crow[q], WS = crow[CR_WS + q];
                float4 U1 = make_float4(0.f, 0.f, 0.f, 0.f), U2 = U1, U3 = U1;
                if (kGrad) U2 = crow[4 + q];
                const float wd[4] = {WD.x, WD.y, WD.z, WD.w}, ws[4] = {WS.x, WS.y, WS.z, WS.w};
                float u1[4] = {U1.x, U1.y, U1.z, U1.w}, u3[4] = {U3.x, U3.y, U3.z, U3.w};
                const float u2[4] = {U2.x, U2.y, U2.z, U2.w};
                if (kGrad) {   // the same products the builder formed for the cell's P sums (cs_math.cuh: cell_band)
#pragma unroll
                    for (int h = 0; h < 4; ++h)
                        if (4 * q + h < NF) { u1[h] = mul_(kc.lnd[4 * q + h], wd[h]); u3[h] = mul_(kc.lns[4 * q + h], ws[h]); }
                }
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int f = 4 * q + h;
                    if (f < NF) {
                        const float2 dq = *reinterpret_cast<const float2 *>(st + (2 * f) * HALF);
                        const float2 du = *reinterpret_cast<const float2 *>(st + (2 * f + 1) * HALF);
                        CellCols<float> C;
                        C.wd = wd[h]; C.u1 = u1[h]; C.u2 = u2[h]; C.ws = ws[h]; C.u3 = u3[h];
                        pix_band<kGrad>(A, C, kc.w[f], dq, du);
                    }
                }
            }
            const float4 S0 = crow[CR_SC], S1 = crow[CR_SC + 1], S3 = crow[CR_SC + 3];
            float4 S2 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (kGrad) S2 = crow[CR_SC + 2];
            CellScal<float> C;
            C.l10 = S0.x; C.l20 = S0.y; C.l21 = S0.z; C.id1 = S0.w; C.id2 = S1.x;
            C.P10 = S1.y; C.P11 = S1.z; C.P12 = S1.w; C.P20 = S2.x; C.P21 = S2.y; C.P22 = S2.z; C.P30 = S2.w;
            C.P31 = S3.x; C.P32 = S3.y; C.bad = S3.z;
            float2 sq[3], su[3], ll;
            float2 t0 = make_float2(0.f, 0.f), t1 = t0, t2 = t0, t3 = t0;
            if (MODE == MODE_CHI2) {   // second pass over the bands while the stages are still held: chi^2 of the residual
                pix_solve(A, C, kc.inv_m00, sq, su, ll);
                float2 xq = make_float2(0.f, 0.f), xu = xq;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 WD = crow[q], WS = crow[CR_WS + q];
                    const float wd[4] = {WD.x, WD.y, WD.z, WD.w}, ws[4] = {WS.x, WS.y, WS.z, WS.w};
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const int f = 4 * q + h;
                        if (f < NF) {
                            const float2 dq = *reinterpret_cast<const float2 *>(st + (2 * f) * HALF);
                            const float2 du = *reinterpret_cast<const float2 *>(st + (2 * f + 1) * HALF);
                            pix_chi2_band(xq, xu, sq, su, wd[h], ws[h], kc.w[f], kc.invw[f], dq, du);
                        }
                    }
                }
                t3 = sel_inf(C.bad, add_(xq, xu));
            }
            __syncwarp();   // every lane has read its data and cell rows: hand the slots back
            if (lane == 0) { mbar_arrive(&empty_d[sd]); mbar_arrive(&empty_c[sc]); }
            if (MODE != MODE_CHI2) pix_solve(A, C, kc.inv_m00, sq, su, ll);
            if (MODE == MODE_VALUE) {
                t3 = ll;
            } else if (MODE == MODE_GRAD) {
                pix_grad_terms(A, C, sq, su, t0, t1, t2);
                t3 = ll;
            } else if (MODE == MODE_CMBVAR) {
                t0 = sq[0]; t1 = su[0]; t2 = mul_(sq[0], sq[0]); t3 = mul_(su[0], su[0]);
            }
            mbar_wait(&empty_t[stt], (uint32_t)(((n / NT) & 1) ^ 1));
            double *tm = sterm + stt * 4 * NCONS;
            if (!ModeTraits<MODE>::region_only) {
                tm[so0] = pair_sum(t0.x, t0.y); tm[so1] = pair_sum(t1.x, t1.y); tm[so2] = pair_sum(t2.x, t2.y);
            }
            tm[so3] = pair_sum(t3.x, t3.y);
            named_arrive(1 + stt, NCONS + 32);
            ++n;
        }
    }
}

}  // namespace cs
