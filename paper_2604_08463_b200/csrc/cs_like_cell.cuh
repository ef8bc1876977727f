// cs_like_cell.cuh -- k_like_cell: the fused per-pixel kernel (a2 + first level of a3, a4, f1) in its "cell" form.
//
// Everything in Eq. 5/6/17 that depends only on the pixel's cluster triple (k0,k1,k2) -- the weighted columns
// N^-1 a_d, N^-1 a_s, N^-1 da_d/dT, the matrix M = A^T N^-1 A, its LDL^T factors and the nine
// contractions P_{theta,c} = sum_f w_f (da_f/dtheta) A_{f,c} -- is the same for all pixels of a tile that share the
// triple (a "cell").  It is hoisted out of the pixel loop: per entry, builder warps evaluate it once per cell of
// the tile into shared memory, and a pixel-eval is left with 12 dot products of length nfreq between its data
// (Q, U) and six weighted columns, two 3x3 triangular solves and a handful of FMAs:
//
//     b_S  = A^T N^-1 d_S                        (3 dots per Stokes)            Eq. 5
//     c_S  = (dA/dtheta)^T N^-1 d_S              (3 dots per Stokes)
//     s_S  = M^-1 b_S  via the cell's LDL^T ;   ll = -1/2 sum_S b_S . s_S       Eq. 5, 6
//     g_th = - sum_S s_{S,c(th)} ( c_{S,th} - sum_c P_{th,c} s_{S,c} )          Eq. 17 with r = d - A s expanded
//
// CTA = 16 warps, one CTA per SM, warp-specialised:
//   warps 0-7    consumers: one pixel of the 256-pixel tile per thread, loop over the group's entries
//   warps 8-10   builders : one cell per thread, fill the cell table of a later entry while earlier ones are consumed
//   warps 11-14  reducers : first level of the ordered fp64 reduction (a3) of the terms the consumers leave behind,
//                           one warp per entry in flight
//   warp  15     loader   : per entry, one TMA box [2*nfreq rows x 256 pixels] into the data ring and the distinct table
//                           rows of the tile's cells (plain loads, one entry ahead) into the row ring
// Every hand-over is an mbarrier pair (full/empty per ring slot): data ring, cell-table ring, term ring.  No role
// ever waits at a CTA-wide barrier after the prologue.
// shared memory: data ring [ND][2*NF][256] | cell tables [NC][CELL_CAP][CSTRIDE] | term ring [NT][4][TROW] |
//                barriers | per-entry meta | segment plan
#pragma once
#include "cs_kernels.cuh"
#include "cs_math.cuh"

namespace cs {

constexpr int NR = 5;        // table-row ring depth: builders run up to NC entries ahead of the consumers, which read
                             // the T_d and beta_s rows of their cell from the same stage (NR >= NC + 2)
template <int NF>
struct DataDepth { static constexpr int value = (NF == 15) ? 3 : 2; };   // data ring depth (entries in flight)
constexpr int RSTRIDE = 20;   // floats per staged table row (16 + 4 pad: consecutive rows start 20 banks apart, no conflicts)
constexpr int NBG = 1;       // builder groups: group g builds the entries i = g (mod NBG)
constexpr int NC = 3;        // cell-table ring depth (a multiple of NBG)
constexpr int NT = 4;        // term ring depth
constexpr int NBUILD = NBG * CELL_CAP;           // builder threads (one per cell and group)
constexpr int NRED = 128;                        // reducer threads
constexpr int CELL_THREADS = TP + NBUILD + NRED + 32;   // 512
static_assert(SEG_MAX <= 4 * CHUNK_LEN && CELL_CAP % 32 == 0 && NC % NBG == 0, "builder warps / ring slots per group");

// cell row layout (floats): [0..15] w a_d per band; [16..31] scalars l10 l20 l21 1/d1 | 1/d2 P10 P11 P12 | P20 P21 P22 P30 |
// P31 P32 bad -.  The other two weighted columns depend on one cluster id only and are formed by the consumers from
// the staged table rows, which many lanes of a warp share: w a_s = w Fs'[k2], w a_d dlnG = dlnG[k1] (w a_d).

template <int NF>
constexpr size_t cell_smem_bytes() {
    constexpr int ND = DataDepth<NF>::value;
    return (size_t)ND * 2 * NF * TP * 4               // data ring
           + (size_t)NR * ROW_CAP * RSTRIDE * 4       // table rows of the tile's cells, staged per entry
           + (size_t)NC * CELL_CAP * CSTRIDE * 4      // cell tables
           + (size_t)NT * 4 * TROW * 4                // term ring
           + (size_t)NT * CHUNK_CAP * 8               // chunk sums of the reducer warps (fp64)
           + (2 * ND + 2 * NC + 2 * NT + 2 * NR) * 8  // mbarriers
           + GROUP_MAX * 16                           // per-entry table base, data row, entry id
           + CHUNK_CAP * (2 + 2 + 4)                  // chunk descriptors, segment descriptors, output slots
           + 16 * 4;                                  // meta
}

// Term-ring "full" hand-over on hardware named barriers 1..NT (consumers arrive, the slot's reducer warp syncs): a
// warp blocked in bar.sync takes no issue slots, unlike a polling mbarrier wait.
__device__ __forceinline__ void terms_arrive(int slot) {
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(slot + 1), "n"(TP + 32) : "memory");
}
__device__ __forceinline__ void terms_wait(int slot) { asm volatile("bar.sync %0, %1;" ::"r"(slot + 1), "n"(TP + 32) : "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Reducer plan of a tile in shared memory: every (term, cluster) segment of <= SEG_MAX rank-ordered terms is cut into
// 1..4 chunks of <= CHUNK_LEN ranks.  s_cdesc[chunk] = start | (len-1) << 8 | term << 11;
// s_sdesc[segment] = first chunk | (chunks-1) << 12; s_slot[segment] = cluster-major slot in the entry's partial row.
template <int MODE>
__device__ __forceinline__ void load_chunk_plan(const MapDev *__restrict__ maps, const CfgDev &cfg, int tile, int tid,
                                                uint16_t *s_cdesc, uint16_t *s_sdesc, int32_t *s_slot, int32_t *meta) {
    constexpr int T0 = ModeTraits<MODE>::region_only ? 3 : 0;
    int sbase = 0, cbase = 0;
#pragma unroll
    for (int t = T0; t < 4; ++t) {
        const MapDev m = maps[(MODE == MODE_CMBVAR) ? cfg.map[3] : cfg.map[t]];
        const int s0 = m.segptr[tile], ns = m.segptr[tile + 1] - s0;
        const int nc = m.chunkptr[tile + 1] - m.chunkptr[tile];
        if (tid < ns) {
            const uint32_t desc = m.segdesc[s0 + tid];
            const int start = desc & 0xff, len = (int)(desc >> 8) + 1;
            const int first = cbase + m.segcfirst[s0 + tid], cnt = (len + CHUNK_LEN - 1) / CHUNK_LEN;
            s_sdesc[sbase + tid] = (uint16_t)(first | ((cnt - 1) << 12));
            s_slot[sbase + tid] = ((MODE == MODE_CMBVAR) ? t * m.nseg : cfg.segbase[t]) + m.segslot[s0 + tid];
            for (int q = 0; q < cnt; ++q) {
                const int l = min(CHUNK_LEN, len - CHUNK_LEN * q);
                s_cdesc[first + q] = (uint16_t)((start + CHUNK_LEN * q) | ((l - 1) << 8) | (t << 11));
            }
        }
        sbase += ns; cbase += nc;
    }
    if (tid == 0) { meta[0] = cbase; meta[1] = sbase; }
}

// First level of the ordered reduction (a3) of one entry by one reducer warp, in fp64 and in a fixed order:
// step 1, one lane per chunk: (x0 + x4) + (x1 + x5) paired with (x2 + x6) + (x3 + x7) over the chunk's <= 8 ranks
// taken in an order rotated by the lane, straight-line so that the lanes do not diverge; step 2, one lane per segment: the
// segment's chunk sums left to right, stored at the segment's cluster-major slot of the entry's partial row.
__device__ __forceinline__ void reduce_entry(const float *tbuf, int lane, const int32_t *meta, const uint16_t *s_cdesc,
                                             const uint16_t *s_sdesc, const int32_t *s_slot, double *csum,
                                             double *__restrict__ prow) {
    const int nchunk = meta[0], nseg = meta[1];
    for (int r = lane; r < nchunk; r += 32) {
        const uint32_t d = s_cdesc[r];
        const int start = d & 0xff, len = (int)((d >> 8) & 7) + 1, t = (int)(d >> 11);
        csum[r] = chunk_sum(tbuf + t * TROW, start, len);   // cs_math.cuh: the same order as the direct kernel's sums
    }
    __syncwarp();
    for (int r = lane; r < nseg; r += 32) {
        const uint32_t d = s_sdesc[r];
        const int first = d & 0xfff, cnt = (int)(d >> 12) + 1;
        double acc = csum[first];
        if (cnt > 1) acc += csum[first + 1];
        if (cnt > 2) acc += csum[first + 2];
        if (cnt > 3) acc += csum[first + 3];
        prow[s_slot[r]] = acc;
    }
    __syncwarp();
}

// The four table rows of a cell (Fd', G, dlnG, Fs'), loaded one entry ahead of their use.
struct CellRows {
    float4 Fd[4], G[4], dG[4], Fs[4];
};
template <bool GRAD>
__device__ __forceinline__ void load_cell_rows(const float *tb, const int4 rows, CellRows &R) {   // tb: staged rows (smem)
    const float4 *rFd = reinterpret_cast<const float4 *>(tb + rows.x * RSTRIDE);
    const float4 *rG = reinterpret_cast<const float4 *>(tb + rows.y * RSTRIDE);
    const float4 *rdG = reinterpret_cast<const float4 *>(tb + rows.z * RSTRIDE);
    const float4 *rFs = reinterpret_cast<const float4 *>(tb + rows.w * RSTRIDE);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        R.Fd[q] = rFd[q]; R.G[q] = rG[q]; R.Fs[q] = rFs[q];
        R.dG[q] = GRAD ? rdG[q] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// One cell (Eq. 2 columns -> weighted column, M, LDL^T, P; cs_math.cuh) from the entry's four table rows.
template <bool GRAD>
__device__ __forceinline__ void build_cell(const CellRows &R, const KConst &kc, float *__restrict__ out, int32_t *err) {
    const float2 *w2 = reinterpret_cast<const float2 *>(kc.w);
    const float2 *lnd2 = reinterpret_cast<const float2 *>(kc.lnd);
    const float2 *lns2 = reinterpret_cast<const float2 *>(kc.lns);
    const float4 *vFd = R.Fd, *vG = R.G, *vdG = R.dG, *vFs = R.Fs;
    CellSums S;
    cell_sums_zero(S);
    float4 *o4 = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float2 wd[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int j = 2 * q + h;
            const float2 Fd = h ? make_float2(vFd[q].z, vFd[q].w) : make_float2(vFd[q].x, vFd[q].y);
            const float2 G = h ? make_float2(vG[q].z, vG[q].w) : make_float2(vG[q].x, vG[q].y);
            const float2 dG = h ? make_float2(vdG[q].z, vdG[q].w) : make_float2(vdG[q].x, vdG[q].y);
            const float2 as = h ? make_float2(vFs[q].z, vFs[q].w) : make_float2(vFs[q].x, vFs[q].y);
            wd[h] = cell_pair<GRAD>(S, Fd, G, dG, as, w2[j], lnd2[j], lns2[j]);
        }
        o4[q] = make_float4(wd[0].x, wd[0].y, wd[1].x, wd[1].y);
    }
    CellScal C;
    cell_finish<GRAD>(S, kc.inv_m00, C);
    if (C.bad != 0.f) atomicOr(err, ERR_SINGULAR);
    o4[4] = make_float4(C.l10, C.l20, C.l21, C.id1);
    o4[5] = make_float4(C.id2, C.P10, C.P11, C.P12);
    o4[6] = make_float4(C.P20, C.P21, C.P22, C.P30);
    o4[7] = make_float4(C.P31, C.P32, C.bad, 0.f);
}

template <int NF, int MODE>
__global__ void __launch_bounds__(CELL_THREADS, 1) k_like_cell(const __grid_constant__ CUtensorMap tmap, const LikeParams P) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int STAGE = 2 * NF * TP;   // floats per data stage
    constexpr int ND = DataDepth<NF>::value;
    float *ring = reinterpret_cast<float *>(smem_raw);
    float *rowbuf = ring + ND * STAGE;
    float *cells = rowbuf + NR * ROW_CAP * RSTRIDE;
    float *sterm = cells + NC * CELL_CAP * CSTRIDE;
    double *csum = reinterpret_cast<double *>(sterm + NT * 4 * TROW);
    uint64_t *bars = reinterpret_cast<uint64_t *>(csum + NT * CHUNK_CAP);
    uint64_t *full_d = bars, *empty_d = bars + ND, *full_c = bars + 2 * ND, *empty_c = bars + 2 * ND + NC;
    uint64_t *full_t = bars + 2 * ND + 2 * NC, *empty_t = full_t + NT;
    uint64_t *full_r = empty_t + NT, *empty_r = full_r + NR;
    const float **s_tab = reinterpret_cast<const float **>(empty_r + NR);
    int32_t *s_drow = reinterpret_cast<int32_t *>(s_tab + GROUP_MAX);
    int32_t *s_ent = s_drow + GROUP_MAX;
    int32_t *s_slot = s_ent + GROUP_MAX;
    int32_t *meta = s_slot + CHUNK_CAP;
    uint16_t *s_cdesc = reinterpret_cast<uint16_t *>(meta + 16);
    uint16_t *s_sdesc = s_cdesc + CHUNK_CAP;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x;
    const Group grp = P.groups[blockIdx.y];
    const CfgDev cfg = P.cfgs[grp.cfg];
    const int64_t npix = P.npix;
    const int nrows = 2 * P.nfreq;
    constexpr bool kReduce = (MODE != MODE_MAPS);
    constexpr bool kGrad = (MODE == MODE_GRAD);

    // ---------------- prologue (all threads) ----------------
    if (tid == 0) {
        for (int s = 0; s < ND; ++s) { mbar_init(&full_d[s], 1); mbar_init(&empty_d[s], TP / 32); }
        for (int s = 0; s < NC; ++s) { mbar_init(&full_c[s], CELL_CAP / 32); mbar_init(&empty_c[s], TP / 32); }
        for (int s = 0; s < NT; ++s) { mbar_init(&full_t[s], TP / 32); mbar_init(&empty_t[s], 1); }
        for (int s = 0; s < NR; ++s) { mbar_init(&full_r[s], 1); mbar_init(&empty_r[s], CELL_CAP / 32 + TP / 32); }   // one builder group + consumers
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    load_group(P, grp, nrows, tid, s_tab, s_drow, s_ent, meta + 12);
    if (kReduce && tid < TP) load_chunk_plan<MODE>(P.maps, cfg, tile, tid, s_cdesc, s_sdesc, s_slot, meta);
    if (NF > 15 && P.nfreq < NF) {   // generic path: rows beyond nfreq are never copied; they must read as zero
        for (int s = 0; s < ND; ++s)
            for (int r = nrows * TP + tid; r < STAGE; r += CELL_THREADS) ring[s * STAGE + r] = 0.f;
    }
    __syncthreads();
    const int count = meta[12] + meta[13];   // entries of the group that are not skipped
    if (count == 0) return;

    if (warp == CELL_THREADS / 32 - 1) {
        // ---------------- loader warp ----------------
        // per entry: (1) the distinct table rows this tile's cells read, loaded one entry ahead by all lanes, into the
        // row ring; (2) the data box into the data ring (one TMA by lane 0, or plain loads when rows of d are not
        // 16-byte aligned)
        const uint32_t box_bytes = (uint32_t)nrows * TP * 4u;
        const int r0 = cfg.rowptr[tile], nrow = cfg.rowptr[tile + 1] - r0;
        constexpr int NQ = ROW_CAP * 4 / 32;   // float4 quarters of rows per lane
        int myoff[NQ];                         // float offset of this lane's k-th quarter inside an entry's table block
#pragma unroll
        for (int k = 0; k < NQ; ++k) {
            const int q = lane + 32 * k;       // quarter q = row (q >> 2), part (q & 3)
            myoff[k] = (q < 4 * nrow) ? cfg.rowlist[r0 + (q >> 2)] * NROW + (q & 3) * 4 : -1;
        }
        float4 v[NQ];
        auto fetch = [&](int i) {
            const float *tb = s_tab[i];
#pragma unroll
            for (int k = 0; k < NQ; ++k)
                if (myoff[k] >= 0) v[k] = __ldg(reinterpret_cast<const float4 *>(tb + myoff[k]));
        };
        const uint64_t policy = P.evict_first ? policy_evict_first() : policy_evict_normal();
        fetch(0);
        for (int i = 0; i < count; ++i) {
            const int sr = i % NR, s = i % ND;
            mbar_wait_relaxed(&empty_r[sr], (uint32_t)(((i / NR) & 1) ^ 1), 250);
            float *dst = rowbuf + sr * ROW_CAP * RSTRIDE;
#pragma unroll
            for (int k = 0; k < NQ; ++k) {
                const int q = lane + 32 * k;   // quarter q = row (q >> 2), part (q & 3)
                if (myoff[k] >= 0) *reinterpret_cast<float4 *>(dst + (q >> 2) * RSTRIDE + (q & 3) * 4) = v[k];
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&full_r[sr]);
            if (i + 1 < count) fetch(i + 1);   // in flight while lane 0 waits for a data slot
            if (P.use_bulk) {
                if (lane == 0) {
                    mbar_wait_relaxed(&empty_d[s], (uint32_t)(((i / ND) & 1) ^ 1), 250);
                    mbar_expect_tx(&full_d[s], box_bytes);
                    tma_box_g2s(ring + s * STAGE, &tmap, tile * TP, s_drow[i], &full_d[s], policy);
                }
            } else {   // rows of d not 16-byte aligned: plain loads by the whole warp
                mbar_wait_relaxed(&empty_d[s], (uint32_t)(((i / ND) & 1) ^ 1), 250);
                const int64_t row0 = s_drow[i];
                for (int r = 0; r < nrows; ++r)
                    for (int x = lane; x < TP; x += 32) {
                        const int64_t px = (int64_t)tile * TP + x;
                        ring[s * STAGE + r * TP + x] = (px < npix) ? P.d[(row0 + r) * npix + px] : 0.f;
                    }
                __syncwarp();
                if (lane == 0) mbar_arrive(&full_d[s]);
            }
        }
        return;
    }
    if (warp >= (TP + NBUILD) / 32) {
        // ---------------- reducer warps: first level of a3, one entry behind the consumers ----------------
        if (!kReduce) return;
        // reducer warp r owns term-ring slot r and the entries i = r (mod NT)
        static_assert(NRED / 32 == NT, "one reducer warp per term-ring slot");
        const int s = warp - (TP + NBUILD) / 32;
        for (int i = s; i < count; i += NT) {
            terms_wait(s);
            reduce_entry(sterm + s * 4 * TROW, lane, meta, s_cdesc, s_sdesc, s_slot, csum + s * CHUNK_CAP,
                         P.partial + (int64_t)s_ent[i] * P.PS);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_t[s]);
        }
        return;
    }
    if (warp >= TP / 32) {
        // ---------------- builder warps: thread c builds cell c of this tile for every entry ----------------
        const int g = (tid - TP) / CELL_CAP, c = (tid - TP) % CELL_CAP;
        const int c0 = cfg.cellptr[tile], ncell = cfg.cellptr[tile + 1] - c0;
        int4 rows = make_int4(0, 0, 0, 0);
        if (c < ncell) rows = *reinterpret_cast<const int4 *>(cfg.cellrows + 4 * (int64_t)(c0 + c));
        for (int i = g; i < count; i += NBG) {
            const int s = i % NC, sr = i % NR;
            CellRows R;
            mbar_wait_relaxed(&full_r[sr], (uint32_t)((i / NR) & 1));
            if (c < ncell) load_cell_rows<kGrad>(rowbuf + sr * ROW_CAP * RSTRIDE, rows, R);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_r[sr]);
            mbar_wait_relaxed(&empty_c[s], (uint32_t)(((i / NC) & 1) ^ 1));
            if (c < ncell) build_cell<kGrad>(R, P.kc, cells + (s * CELL_CAP + c) * CSTRIDE, P.err);
            __syncwarp();
            if (lane == 0) mbar_arrive(&full_c[s]);
        }
        return;
    }

    // ---------------- consumers ----------------
    const int64_t p = (int64_t)tile * TP + tid;
    int so0 = 0 * TROW + TP, so1 = 1 * TROW + TP, so2 = 2 * TROW + TP, so3 = 3 * TROW + TP;
    int cid = 0xFF;
    if (p < npix) {
        cid = cfg.cellid[p];
        if (kReduce) {
            const int m3 = cfg.map[3];
            if (MODE == MODE_CMBVAR) {
                const int r = P.maps[m3].rank[p];
                so0 = 0 * TROW + r; so1 = 1 * TROW + r; so2 = 2 * TROW + r; so3 = 3 * TROW + r;
            } else {
                if (kGrad) {   // a pixel masked in another map still owns a rank here: its slot must read 0
                    if (P.maps[cfg.map[0]].idx[p] >= 0) so0 = 0 * TROW + P.maps[cfg.map[0]].rank[p];
                    if (P.maps[cfg.map[1]].idx[p] >= 0) so1 = 1 * TROW + P.maps[cfg.map[1]].rank[p];
                    if (P.maps[cfg.map[2]].idx[p] >= 0) so2 = 2 * TROW + P.maps[cfg.map[2]].rank[p];
                }
                so3 = 3 * TROW + P.maps[m3].rank[p];
            }
        }
    }
    const bool live = cid != 0xFF;
    int slot_dg = 0, slot_fs = 0;   // slots of this pixel's dlnG[k1] and Fs'[k2] rows in the tile's staged row list
    if (live) {
        const int32_t *cr = cfg.cellrows + 4 * (int64_t)(cfg.cellptr[tile] + cid);
        slot_dg = cr[2] * RSTRIDE; slot_fs = cr[3] * RSTRIDE;
    }
    const float2 *w2 = reinterpret_cast<const float2 *>(P.kc.w);
    const float2 *lnd2 = reinterpret_cast<const float2 *>(P.kc.lnd);
    const float2 *lns2 = reinterpret_cast<const float2 *>(P.kc.lns);
    const float inv_m00 = P.kc.inv_m00;

    for (int i = 0; i < count; ++i) {
        const int sd = i % ND, sc = i % NC, sr = i % NR;
        mbar_wait(&full_c[sc], (uint32_t)((i / NC) & 1));   // the builders waited for full_r[sr]: the rows are there too
        mbar_wait(&full_d[sd], (uint32_t)((i / ND) & 1));
        PixSums A;
        pix_sums_zero(A);
        float4 S0 = make_float4(0.f, 0.f, 0.f, 0.f), S1 = S0, S2 = S0, S3 = S0;
        float chi = 0.f;
        if (live) {
            const float *st = ring + sd * STAGE + tid;
            const float4 *cell = reinterpret_cast<const float4 *>(cells + (sc * CELL_CAP + cid) * CSTRIDE);
            const float4 *rfs = reinterpret_cast<const float4 *>(rowbuf + sr * ROW_CAP * RSTRIDE + slot_fs);
            const float4 *rdg = reinterpret_cast<const float4 *>(rowbuf + sr * ROW_CAP * RSTRIDE + slot_dg);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 WD = cell[q], FS = rfs[q];
                float4 DG = make_float4(0.f, 0.f, 0.f, 0.f);
                if (kGrad) DG = rdg[q];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int j = 2 * q + h;
                    const float2 dq = make_float2(st[(4 * j + 0) * TP], (2 * j + 1 < NF) ? st[(4 * j + 2) * TP] : 0.f);
                    const float2 du = make_float2(st[(4 * j + 1) * TP], (2 * j + 1 < NF) ? st[(4 * j + 3) * TP] : 0.f);
                    const float2 wd = h ? make_float2(WD.z, WD.w) : make_float2(WD.x, WD.y);
                    const float2 fs = h ? make_float2(FS.z, FS.w) : make_float2(FS.x, FS.y);
                    const float2 dg = h ? make_float2(DG.z, DG.w) : make_float2(DG.x, DG.y);
                    pix_pair<kGrad>(A, wd, fs, dg, w2[j], lnd2[j], lns2[j], dq, du);   // cs_math.cuh
                }
            }
            S0 = cell[4]; S1 = cell[5];
            if (kGrad) S2 = cell[6];
            S3 = cell[7];
            if (MODE == MODE_CHI2) {   // second pass over the bands while the stages are still held: chi^2 of the residual
                CellScal C;
                C.l10 = S0.x; C.l20 = S0.y; C.l21 = S0.z; C.id1 = S0.w; C.id2 = S1.x; C.bad = S3.z;
                C.P10 = C.P11 = C.P12 = C.P20 = C.P21 = C.P22 = C.P30 = C.P31 = C.P32 = 0.f;
                float sq[3], su[3], ll;
                pix_solve(A, C, inv_m00, sq, su, ll);
                const float2 *iw2 = reinterpret_cast<const float2 *>(P.kc.invw);
                ChiCoef K;
                chi_coef(sq, su, K);
                ChiSums X;
                X.q = X.u = make_float2(0.f, 0.f);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 WD = cell[q], FS = rfs[q];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int j = 2 * q + h;
                        const float2 dq = make_float2(st[(4 * j + 0) * TP], (2 * j + 1 < NF) ? st[(4 * j + 2) * TP] : 0.f);
                        const float2 du = make_float2(st[(4 * j + 1) * TP], (2 * j + 1 < NF) ? st[(4 * j + 3) * TP] : 0.f);
                        const float2 wd = h ? make_float2(WD.z, WD.w) : make_float2(WD.x, WD.y);
                        const float2 fs = h ? make_float2(FS.z, FS.w) : make_float2(FS.x, FS.y);
                        pix_chi2_pair(X, K, wd, fs, w2[j], iw2[j], dq, du);
                    }
                }
                chi = (C.bad != 0.f) ? CUDART_INF_F : hsum(X.q) + hsum(X.u);
            }
        }
        __syncwarp();   // every lane has read its data and cell rows: hand the slots back
        if (lane == 0) { mbar_arrive(&empty_d[sd]); mbar_arrive(&empty_c[sc]); mbar_arrive(&empty_r[sr]); }

        float t0 = 0.f, t1 = 0.f, t2 = 0.f, t3 = 0.f;
        if (live) {
            CellScal C;
            C.l10 = S0.x; C.l20 = S0.y; C.l21 = S0.z; C.id1 = S0.w; C.id2 = S1.x;
            C.P10 = S1.y; C.P11 = S1.z; C.P12 = S1.w; C.P20 = S2.x; C.P21 = S2.y; C.P22 = S2.z; C.P30 = S2.w;
            C.P31 = S3.x; C.P32 = S3.y; C.bad = S3.z;
            float sq[3], su[3], ll;
            if (MODE != MODE_CHI2) pix_solve(A, C, inv_m00, sq, su, ll);
            if (MODE == MODE_VALUE) {
                t3 = ll;
            } else if (MODE == MODE_CHI2) {
                t3 = chi;
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
        if (kReduce) {
            const int st = i % NT;
            mbar_wait(&empty_t[st], (uint32_t)(((i / NT) & 1) ^ 1));
            float *tm = sterm + st * 4 * TROW;
            if (!ModeTraits<MODE>::region_only) { tm[so0] = t0; tm[so1] = t1; tm[so2] = t2; }
            tm[so3] = t3;
            terms_arrive(st);
        }
    }
}

}  // namespace cs
