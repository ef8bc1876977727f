// cs_lib.cu -- C ABI of libcs (include/cs.h): context, layouts and reduction plans, launches.  No CPU compute path
// exists: every arithmetic step of the hot path runs in the kernels of cs_tables.cuh / cs_like_sc.cuh /
// cs_like_direct.cuh / cs_optim.cuh; the host code below only validates, builds index structures once per clustering
// and launches.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>
#include <stdexcept>
#include <new>
#include <vector>

#include "../../include/cs.h"
#include "cs_tables.cuh"
#include "cs_like_sc.cuh"
#include "cs_like_direct.cuh"
#include "cs_optim.cuh"
#include "cs_cells.cuh"
#include "cs_kmeans.cuh"

using namespace cs;

#define CK(call)                                   \
    do {                                           \
        cudaError_t err__ = (call);                \
        if (err__ != cudaSuccess) return CS_ECUDA; \
    } while (0)

// No exception may cross the C ABI: host-side plan building allocates std::vectors.
#define CS_GUARD_BEGIN try {
#define CS_GUARD_END                                  \
    }                                                 \
    catch (const std::bad_alloc &) { return CS_ENOMEM; } \
    catch (...) { return CS_EINVAL; }

namespace {

struct MapHost {
    int32_t K = 0, nseg = 0;
    int32_t *idx = nullptr;
    uint16_t *rank = nullptr;
    int32_t *segptr = nullptr;
    uint16_t *segdesc = nullptr;
    int32_t *segslot = nullptr;
    int32_t *ksegptr = nullptr;
    int32_t *chunkptr = nullptr;
    uint16_t *segcfirst = nullptr;
};

// Device arrays of one configuration's sorted layout (empty when it stays in place).
struct SortedHost {
    uint32_t *hdr = nullptr;
    int32_t *hdrptr = nullptr;
    uint8_t *cellid = nullptr;
    int32_t *cellptr = nullptr;
    int32_t *cellrows = nullptr;
    int32_t *pospix = nullptr;
};

// Device arrays of one configuration's global cell list (f3; sorted configurations only).
struct CellsHost {
    int32_t *cellpos = nullptr, *celllen = nullptr, *cellreg = nullptr;
    int32_t *kptr[4] = {nullptr, nullptr, nullptr, nullptr}, *klist[4] = {nullptr, nullptr, nullptr, nullptr};
    int32_t ncell = 0;
};

template <typename T>
int dev_upload(T **dst, const std::vector<T> &src, int64_t *bytes) {
    *dst = nullptr;
    size_t n = std::max<size_t>(src.size(), 1) * sizeof(T);
    if (cudaMalloc((void **)dst, n) != cudaSuccess) return CS_ENOMEM;
    if (!src.empty() && cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
        return CS_ECUDA;
    *bytes += (int64_t)n;
    return CS_OK;
}

// Device memory of cs_set_clusters: a clustering scan sets a thousand configurations of some thirty arrays each, so the
// arrays are carved out of 64-MB chunks instead of one cudaMalloc apiece.
struct Arena {
    std::vector<void *> chunks;
    char *cur = nullptr;
    size_t left = 0;
    void *alloc(size_t n) {
        n = (std::max<size_t>(n, 1) + 255) & ~(size_t)255;
        if (n > left) {
            const size_t sz = std::max<size_t>(n, (size_t)64 << 20);
            void *p = nullptr;
            if (cudaMalloc(&p, sz) != cudaSuccess) { cudaGetLastError(); return nullptr; }
            chunks.push_back(p);
            cur = (char *)p; left = sz;
        }
        void *r = cur;
        cur += n; left -= n;
        return r;
    }
    void release() {
        for (void *p : chunks) cudaFree(p);
        chunks.clear(); cur = nullptr; left = 0;
    }
};
template <typename T>
int arena_upload(Arena &ar, T **dst, const std::vector<T> &src, int64_t *bytes) {
    *dst = (T *)ar.alloc(src.size() * sizeof(T));
    if (!*dst) return CS_ENOMEM;
    if (!src.empty() && cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return CS_ECUDA;
    *bytes += (int64_t)((std::max<size_t>(src.size() * sizeof(T), 1) + 255) & ~(size_t)255);
    return CS_OK;
}

}  // namespace

struct cs_ctx {
    // model
    int32_t nfreq = 0, units = 0;
    int64_t npix = 0;
    int32_t ntile_ring = 0;
    int32_t nsm = 1;
    double freqs[NROW] = {0};
    double nu0d = 0, nu0s = 0, tcmb = 0;
    TConst tc;
    KConst kc;
    bool have_ninv = false;
    // options (cs_set_option)
    int32_t opt_layout = CS_LAYOUT_AUTO, opt_form = CS_FORM_AUTO, opt_pixbeta = CS_PIXBETA_AUTO;
    double opt_min_fill = 0.36;         // measured crossover of the two kernels (bench.py cellsweep)
    int64_t opt_copy_limit = 0;         // bytes, 0 = 70 % of the free device memory when the batch is set
    // clusters
    int32_t nmap = 0, ncfg = 0, nregion = 1;
    std::vector<MapHost> maps;          // nmap pixel-space maps, the region pseudo-map, then 4 per sorted configuration
    std::vector<CfgDev> cfgs;
    std::vector<SortedHost> sorted;     // ncfg
    std::vector<CellsHost> cellsh;      // ncfg
    CellsDev *d_cells = nullptr;
    int32_t ncell_max = 0;
    std::vector<int32_t> npix_live;     // [ncfg*nregion]
    MapDev *d_maps = nullptr;
    CfgDev *d_cfgs = nullptr;
    int32_t *d_npix_live = nullptr;
    int64_t cluster_bytes = 0;
    Arena cl_arena;                     // every device array of cs_set_clusters
    // data
    const float *d = nullptr;
    int32_t ndata = 0;
    CUtensorMap tmap;                   // d as [ndata*2*nfreq, npix], box [2*nfreq, 256]
    bool have_tmap = false;
    // batch
    int32_t batch = 0, ktot_max = 0;
    int32_t nrun_sc = 0, nrun_dir = 0;  // d_runs = [sorted-cell runs | direct runs]
    int64_t W_sc = 0, W_dir = 0;
    int64_t nparam = 0, nrows = 0, PS = 0;
    std::vector<int32_t> cfg_of, data_of, elist;
    std::vector<int64_t> param_off, copy_off, tab_off;
    std::vector<PosInfo> pinfo;         // per position of elist
    std::vector<Run> runs;
    std::vector<CopyJob> jobs;          // private copies of the sorted layout, ordered by data set
    std::vector<int64_t> cfg_tstride;   // [ncfg] floats between consecutive tiles of a configuration's copies in this batch
    int32_t *d_cfg_of = nullptr, *d_data_of = nullptr, *d_elist = nullptr;
    int64_t *d_param_off = nullptr, *d_tab_off = nullptr;
    TabBlock *d_tabblk = nullptr;      // k_tables' work list: blocks of TAB_ROWS_PER_BLOCK parameters of every entry
    int64_t ntabblk = 0;
    MergeBlock *d_mblk = nullptr;      // k_merge's work list: [region blocks of every entry | cluster blocks of every entry]
    int64_t nmblk_region = 0, nmblk_all = 0;
    PosInfo *d_pinfo = nullptr;
    Run *d_runs = nullptr;
    CopyJob *d_jobs = nullptr;
    float *d_tab = nullptr, *d_copy = nullptr;
    double *d_pcopy = nullptr;          // the parameters the tables were last built from
    bool any_pixbeta = false;           // some entry of the batch reads d_pcopy (per-pixel beta_d); else it is not filled
    double *d_partial = nullptr;
    int64_t batch_bytes = 0, copy_bytes = 0;
    int32_t job_ntile_max = 0;
    // selections of cs_component_maps: small pinned staging ring, so that the call stays asynchronous
    static constexpr int SEL_RING = 4;
    int32_t *h_sel = nullptr;           // pinned [SEL_RING][sel_cap] ints (entry list, then runs)
    int32_t *d_sel = nullptr;           // device  [SEL_RING][sel_cap]
    int64_t sel_cap = 0;
    cudaEvent_t sel_ev[SEL_RING] = {nullptr, nullptr, nullptr, nullptr};
    int64_t sel_n = 0;
    // f3 workspace (cs_cell_moments)
    double *d_mom = nullptr, *d_ccout = nullptr;
    int64_t *d_mom_off = nullptr;
    MomJob *d_momjobs = nullptr;
    float *d_w = nullptr;
    int64_t cc_bytes = 0, cc_out_stride = 0;
    bool have_moments = false;
    // optimizer workspace
    OptWork opt;
    int64_t opt_bytes = 0;
    // host-eval staging
    float *d_stage = nullptr;
    int64_t stage_bytes = 0;
    double *d_hparams = nullptr, *d_hnll = nullptr, *d_hgrad = nullptr;
    Run *d_hruns = nullptr;
    int64_t hruns_cap = 0;
    int64_t hbuf_bytes = 0;
    cudaStream_t copy_stream = nullptr, comp_stream = nullptr;
    // optional timing of the fused kernel (cs_profile): ring of event pairs recorded around every gradient-mode launch
    static constexpr int PROF_RING = 512;
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_ev;   // 2*PROF_RING
    int64_t prof_n = 0;
    // misc
    int32_t *d_err = nullptr;
    TConst *d_tc = nullptr;             // device copy of tc (k_tables stages it in shared memory)
    int64_t launches = 0;
    const int32_t *skip = nullptr;      // set by cs_optimize around line-search trials: entries that already accepted
    bool tables_built = false;
};

namespace {

void free_clusters(cs_ctx *c) {
    c->cl_arena.release();   // every device array of the maps, the sorted layouts, the cell lists and the tables of them
    c->maps.clear();
    c->sorted.clear();
    c->cellsh.clear();
    c->d_cells = nullptr;
    c->ncell_max = 0;
    c->d_maps = nullptr; c->d_cfgs = nullptr; c->d_npix_live = nullptr;
    c->cfgs.clear();
    c->nmap = c->ncfg = 0;
    c->cluster_bytes = 0;
}

void free_opt(cs_ctx *c) {
    opt_free(c->opt);
    c->opt_bytes = 0;
}

void free_batch(cs_ctx *c) {
    cudaFree(c->d_cfg_of); cudaFree(c->d_data_of); cudaFree(c->d_elist);
    cudaFree(c->d_param_off); cudaFree(c->d_tab_off); cudaFree(c->d_tabblk); cudaFree(c->d_mblk); cudaFree(c->d_pinfo); cudaFree(c->d_runs); cudaFree(c->d_jobs);
    cudaFree(c->d_tab); cudaFree(c->d_partial); cudaFree(c->d_copy); cudaFree(c->d_pcopy);
    c->d_pcopy = nullptr;
    c->d_cfg_of = c->d_data_of = c->d_elist = nullptr;
    c->d_param_off = c->d_tab_off = nullptr; c->d_pinfo = nullptr; c->d_tabblk = nullptr; c->ntabblk = 0; c->d_mblk = nullptr; c->nmblk_region = c->nmblk_all = 0;
    c->d_runs = nullptr; c->d_jobs = nullptr;
    c->d_tab = nullptr; c->d_partial = nullptr; c->d_copy = nullptr;
    c->batch = 0; c->nrun_sc = c->nrun_dir = 0; c->batch_bytes = 0; c->copy_bytes = 0;
    c->tables_built = false;
    cudaFree(c->d_hparams); cudaFree(c->d_hnll); cudaFree(c->d_hgrad); cudaFree(c->d_hruns);
    c->d_hparams = c->d_hnll = c->d_hgrad = nullptr; c->d_hruns = nullptr; c->hruns_cap = 0;
    c->hbuf_bytes = 0;
    cudaFree(c->d_mom); cudaFree(c->d_ccout); cudaFree(c->d_mom_off); cudaFree(c->d_momjobs); cudaFree(c->d_w);
    c->d_mom = c->d_ccout = nullptr; c->d_mom_off = nullptr; c->d_momjobs = nullptr; c->d_w = nullptr;
    c->cc_bytes = 0; c->have_moments = false;
    if (c->h_sel) cudaFreeHost(c->h_sel);
    cudaFree(c->d_sel);
    c->h_sel = nullptr; c->d_sel = nullptr; c->sel_cap = 0;
    free_opt(c);
}

// K_RJ -> K_CMB factor u(nu) = (e^x - 1)^2 / (x^2 e^x), x = h nu / (k_B T_cmb)   (R2)
double krj2kcmb(double nu_ghz, double tcmb, double hk) {
    const double x = hk * nu_ghz / tcmb;
    const double em1 = std::expm1(x);
    return em1 * em1 / (x * x * std::exp(x));
}

// Reduction plan of one term map in position space: per tile the rank of every position in the (cluster, position)
// order, that order cut into segments of <= SEG_MAX positions of one cluster, plus the CSR cluster -> segments.
struct MapPlanHost {   // the reduction plan of one term map on the host: computed (on a worker thread), then uploaded
    std::vector<int32_t> idx, segptr, segslot, ksegptr, chunkptr;
    std::vector<uint16_t> rank, segdesc, segcfirst;
    int32_t K = 0, nseg = 0;
};
void compute_map_plan(const int32_t *idx, int32_t K, int64_t npos, int32_t ntile, MapPlanHost &mp) {
    std::vector<uint16_t> &rank = mp.rank;
    rank.assign((size_t)ntile * TPX, (uint16_t)NORANK);
    std::vector<int32_t> &segptr = mp.segptr;
    segptr.assign(ntile + 1, 0);
    std::vector<uint16_t> &segdesc = mp.segdesc;
    segdesc.clear();
    std::vector<int32_t> segcluster;
    segdesc.reserve((size_t)ntile * 16);
    segcluster.reserve((size_t)ntile * 16);
    std::vector<std::pair<int32_t, int32_t>> tmp;
    std::vector<std::pair<uint16_t, int32_t>> tseg;   // (descriptor, cluster)
    std::vector<int32_t> &chunkptr = mp.chunkptr;
    chunkptr.assign(ntile + 1, 0);
    std::vector<uint16_t> &segcfirst = mp.segcfirst;
    segcfirst.clear();
    int32_t nchunk = 0;
    tmp.reserve(TPX);
    for (int32_t t = 0; t < ntile; ++t) {
        tmp.clear();
        const int64_t p0 = (int64_t)t * TPX;
        const int nv = (int)std::min<int64_t>(TPX, npos - p0);
        for (int j = 0; j < nv; ++j)
            if (idx[p0 + j] >= 0) tmp.emplace_back(idx[p0 + j], j);
        std::sort(tmp.begin(), tmp.end());
        segptr[t] = (int32_t)segdesc.size();
        // segments of this tile, longest first: the threads of the reduce phase then walk runs of similar length
        tseg.clear();
        size_t i = 0;
        while (i < tmp.size()) {
            size_t j = i;
            while (j < tmp.size() && tmp[j].first == tmp[i].first && j - i < (size_t)SEG_MAX) ++j;
            tseg.push_back({(uint16_t)(i | ((j - i - 1) << 9)), tmp[i].first});
            i = j;
        }
        std::stable_sort(tseg.begin(), tseg.end(), [](const std::pair<uint16_t, int32_t> &a, const std::pair<uint16_t, int32_t> &b) {
            return (a.first >> 9) > (b.first >> 9);
        });
        chunkptr[t] = nchunk;
        int32_t local = 0;
        for (auto &sg : tseg) {
            segdesc.push_back(sg.first); segcluster.push_back(sg.second);
            segcfirst.push_back((uint16_t)local);
            local += ((sg.first >> 9) + 1 + CHUNK_LEN - 1) / CHUNK_LEN;
        }
        nchunk += local;
        for (size_t q = 0; q < tmp.size(); ++q) rank[p0 + tmp[q].second] = (uint16_t)q;
    }
    segptr[ntile] = (int32_t)segdesc.size();
    chunkptr[ntile] = nchunk;
    const int32_t nseg = (int32_t)segdesc.size();
    // cluster-major slots: the segments of cluster k occupy [ksegptr[k], ksegptr[k+1]) in ascending (tile, chunk) order
    std::vector<int32_t> &ksegptr = mp.ksegptr, &segslot = mp.segslot;
    ksegptr.assign(K + 1, 0);
    segslot.assign(nseg, 0);
    for (int32_t s = 0; s < nseg; ++s) ksegptr[segcluster[s] + 1]++;
    for (int32_t k = 0; k < K; ++k) ksegptr[k + 1] += ksegptr[k];
    std::vector<int32_t> fill(ksegptr.begin(), ksegptr.end() - 1);
    for (int32_t s = 0; s < nseg; ++s) segslot[s] = fill[segcluster[s]]++;
    mp.idx.assign((size_t)ntile * TPX, -1);
    std::copy(idx, idx + npos, mp.idx.begin());
    mp.K = K; mp.nseg = nseg;
}
int upload_map_plan(Arena &ar, const MapPlanHost &mp, MapHost *out, int64_t *bytes) {
    out->K = mp.K; out->nseg = mp.nseg;
    int rc;
    if ((rc = arena_upload(ar, &out->idx, mp.idx, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->rank, mp.rank, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->segptr, mp.segptr, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->segdesc, mp.segdesc, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->segslot, mp.segslot, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->ksegptr, mp.ksegptr, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->chunkptr, mp.chunkptr, bytes))) return rc;
    if ((rc = arena_upload(ar, &out->segcfirst, mp.segcfirst, bytes))) return rc;
    return CS_OK;
}

// Sorted layout of one configuration (cs_internal.h): the live pixels grouped into cells (k0, k1, k2, region), cells
// ordered so that neighbours in the order are neighbours on the sky (by the first pixel of their beta_d cluster, then
// by their own first pixel), every cell padded to an even number of positions, tiles closed early when they would
// hold more than CELL_CAP cells.  Fills the position-space arrays; returns the fill fraction live / (ntile * TPX).
struct SortedPlan {
    std::vector<int32_t> pospix, idx[4], cellptr, cellrows;
    std::vector<int32_t> cellpos, celllen, cellkey[4];   // per tile-cell: first position, live + odd-pad positions, ids
    std::vector<uint8_t> cellid;
    int32_t ntile = 0;
    double fill = 0.0;
};
void plan_sorted(const int32_t *i0, const int32_t *i1, const int32_t *i2, const int32_t *reg, const int32_t K[3], int64_t npix,
                 SortedPlan &sp) {
    struct Px { int32_t a, b, c, r, p; };
    std::vector<Px> px;
    px.reserve((size_t)npix);
    for (int64_t p = 0; p < npix; ++p)
        if (i0[p] >= 0 && i1[p] >= 0 && i2[p] >= 0) px.push_back(Px{i0[p], i1[p], i2[p], reg[p], (int32_t)p});
    std::sort(px.begin(), px.end(), [](const Px &x, const Px &y) {
        if (x.a != y.a) return x.a < y.a;
        if (x.b != y.b) return x.b < y.b;
        if (x.c != y.c) return x.c < y.c;
        if (x.r != y.r) return x.r < y.r;
        return x.p < y.p;
    });
    struct Cell { int32_t first, count, kmin, a, minp; };
    std::vector<Cell> cells;
    std::vector<int32_t> kmin(K[0], INT32_MAX);
    for (size_t i = 0; i < px.size();) {
        size_t j = i;
        while (j < px.size() && px[j].a == px[i].a && px[j].b == px[i].b && px[j].c == px[i].c && px[j].r == px[i].r) ++j;
        cells.push_back(Cell{(int32_t)i, (int32_t)(j - i), 0, px[i].a, px[i].p});
        kmin[px[i].a] = std::min(kmin[px[i].a], px[i].p);
        i = j;
    }
    for (auto &ce : cells) ce.kmin = kmin[ce.a];
    std::sort(cells.begin(), cells.end(), [](const Cell &x, const Cell &y) {
        if (x.kmin != y.kmin) return x.kmin < y.kmin;
        if (x.a != y.a) return x.a < y.a;
        return x.minp < y.minp;
    });
    sp.pospix.clear(); sp.cellid.clear(); sp.cellptr.assign(1, 0); sp.cellrows.clear();
    sp.cellpos.clear(); sp.celllen.clear();
    for (int t = 0; t < 4; ++t) sp.cellkey[t].clear();
    for (int t = 0; t < 4; ++t) sp.idx[t].clear();
    int pos = 0, ncell = 0;   // inside the current tile
    Px last{0, 0, 0, 0, -1};
    auto put = [&](const Px &q, int32_t pix) {
        sp.pospix.push_back(pix);
        sp.idx[0].push_back(q.a); sp.idx[1].push_back(q.b); sp.idx[2].push_back(q.c); sp.idx[3].push_back(q.r);
        if (pos & 1) sp.cellid.push_back((uint8_t)(ncell - 1));
        ++pos;
    };
    auto close_tile = [&]() {
        while (pos < TPX) put(last, -1);   // trailing pads belong to the tile's last cell
        sp.cellptr.push_back((int32_t)(sp.cellrows.size() / 4));
        pos = 0; ncell = 0;
    };
    for (const Cell &ce : cells) {
        int32_t done = 0;
        const int32_t padded = ce.count + (ce.count & 1);
        while (done < padded) {
            if (pos == TPX || ncell == CELL_CAP) close_tile();
            const int32_t take = std::min(padded - done, TPX - pos);
            const Px &q0 = px[ce.first];
            ++ncell;
            sp.cellrows.push_back(q0.a); sp.cellrows.push_back(K[0] + q0.b); sp.cellrows.push_back(K[0] + K[1] + q0.b);
            sp.cellrows.push_back(K[0] + 2 * K[1] + q0.c);
            sp.cellpos.push_back((int32_t)sp.pospix.size()); sp.celllen.push_back(take);
            sp.cellkey[0].push_back(q0.a); sp.cellkey[1].push_back(q0.b); sp.cellkey[2].push_back(q0.c); sp.cellkey[3].push_back(q0.r);
            last = q0;
            for (int32_t j = 0; j < take; ++j) {
                const int32_t src = done + j;
                put(q0, src < ce.count ? px[ce.first + src].p : -1);
            }
            done += take;
        }
    }
    if (pos > 0 || sp.cellptr.size() == 1) {
        if (ncell == 0) {   // no live pixel at all: one dummy cell reading the first table rows, all pads
            sp.cellrows.push_back(0); sp.cellrows.push_back(K[0]); sp.cellrows.push_back(K[0] + K[1]); sp.cellrows.push_back(K[0] + 2 * K[1]);
            sp.cellpos.push_back((int32_t)sp.pospix.size()); sp.celllen.push_back(0);
            for (int t = 0; t < 4; ++t) sp.cellkey[t].push_back(0);
            ncell = 1;
            last = Px{0, 0, 0, 0, -1};
        }
        close_tile();
    }
    sp.ntile = (int32_t)sp.cellptr.size() - 1;
    sp.fill = (double)px.size() / ((double)sp.ntile * TPX);
}

// Tile headers of one sorted configuration (cs_internal.h "tile header"): everything the roles of k_like_sc need to
// know about a tile, packed so that the loader warp fetches it with one bulk copy one tile ahead.
void pack_tile_headers(const SortedPlan &sp, const MapPlanHost (&mp)[4], const int32_t segbase[4], int32_t nseg_region,
                       std::vector<int32_t> &hdrptr, std::vector<uint32_t> &blob) {
    hdrptr.assign(sp.ntile + 1, 0);
    blob.clear();
    for (int32_t tile = 0; tile < sp.ntile; ++tile) {
        const size_t base = blob.size();   // in 32-bit words
        hdrptr[tile] = (int32_t)(base / 4);
        const int32_t c0 = sp.cellptr[tile], ncell = sp.cellptr[tile + 1] - c0;
        int32_t nchunk[4], nseg[4], ctot = 0, stot = 0;
        for (int t = 0; t < 4; ++t) {
            nchunk[t] = mp[t].chunkptr[tile + 1] - mp[t].chunkptr[tile];
            nseg[t] = mp[t].segptr[tile + 1] - mp[t].segptr[tile];
            ctot += nchunk[t]; stot += nseg[t];
        }
        const int32_t off_cells = HDR_META + HDR_CONS;                      // words
        const int32_t off_slot = off_cells + 4 * ncell;
        const int32_t off_cdesc = off_slot + stot;                          // u16 arrays, packed two per word
        const int32_t off_sdesc = off_cdesc + (ctot + 1) / 2;
        const int32_t total = (off_sdesc + (stot + 1) / 2 + 3) & ~3;        // multiple of 16 bytes
        if (total > HDR_CAP_WORDS || ncell > CELL_CAP) throw std::length_error("tile header");   // cannot happen: the caps follow from CELL_CAP
        blob.resize(base + total, 0u);
        uint32_t *h = blob.data() + base;
        h[HM_NCELL] = (uint32_t)ncell; h[HM_NCHUNK] = (uint32_t)ctot; h[HM_NSEG] = (uint32_t)stot;
        h[HM_CBASE3] = (uint32_t)(ctot - nchunk[3]); h[HM_SBASE3] = (uint32_t)(stot - nseg[3]);
        h[HM_NSEGREG] = (uint32_t)nseg_region; h[HM_SEGBASE3] = (uint32_t)segbase[3];
        h[HM_OFF_SLOT] = (uint32_t)off_slot; h[HM_OFF_CDESC] = (uint32_t)off_cdesc; h[HM_OFF_SDESC] = (uint32_t)off_sdesc;
        for (int tid = 0; tid < NCONS; ++tid) {
            const size_t pos = (size_t)tile * TPX + 2 * tid;
            uint32_t r[4];
            for (int t = 0; t < 4; ++t) r[t] = (uint32_t)(mp[t].rank[pos] >> 1) & 0xffu;
            h[HDR_META + 2 * tid] = (uint32_t)sp.cellid[(size_t)tile * NCONS + tid] | (r[0] << 8) | (r[1] << 16) | (r[2] << 24);
            h[HDR_META + 2 * tid + 1] = r[3];
        }
        for (int32_t q = 0; q < 4 * ncell; ++q) h[off_cells + q] = (uint32_t)sp.cellrows[(size_t)4 * c0 + q];
        uint16_t *cdesc = reinterpret_cast<uint16_t *>(h + off_cdesc), *sdesc = reinterpret_cast<uint16_t *>(h + off_sdesc);
        int32_t sb = 0, cb = 0;
        for (int t = 0; t < 4; ++t) {   // the same plan sc_load_plan used to assemble per tile in the kernel
            const int32_t s0 = mp[t].segptr[tile];
            for (int32_t i = 0; i < nseg[t]; ++i) {
                const uint32_t desc = mp[t].segdesc[s0 + i];
                const int start = desc & 0x1ff, len = (int)(desc >> 9) + 1;
                const int first = cb + mp[t].segcfirst[s0 + i], cnt = (len + CHUNK_LEN - 1) / CHUNK_LEN;
                sdesc[sb + i] = (uint16_t)((start >> 1) | ((cnt - 1) << 8) | (t << 10));
                h[off_slot + sb + i] = (uint32_t)(segbase[t] + mp[t].segslot[s0 + i]);
                for (int q = 0; q < cnt; ++q) {
                    const int l = std::min(CHUNK_LEN, len - CHUNK_LEN * q);
                    cdesc[first + q] = (uint16_t)(((start + CHUNK_LEN * q) >> 1) | ((l / 2 - 1) << 8) | (t << 10));
                }
            }
            sb += nseg[t]; cb += nchunk[t];
        }
    }
    hdrptr[sp.ntile] = (int32_t)(blob.size() / 4);
}

// Runs fn(i) for i in [0, n) on the host's threads (plan building is pure host work, independent per map and per
// configuration: a clustering scan sets a thousand configurations).  Returns CS_OK, or what the first call that threw
// stands for: CS_ENOMEM (bad_alloc, or a vector asked for more than it can hold) or CS_EINVAL.  A thread that cannot be
// started is not an error: the calling thread and the ones that did start share the work.
template <class F>
int parallel_for(int n, F fn) {
    const int nt = std::max(1, std::min<int>(n, std::min<unsigned>(16u, std::thread::hardware_concurrency())));
    std::atomic<int> next{0};
    std::atomic<int> rc{CS_OK};
    auto work = [&]() {
        int mine = CS_OK;
        try {
            for (int i = next.fetch_add(1); i < n; i = next.fetch_add(1)) fn(i);
        } catch (const std::bad_alloc &) { mine = CS_ENOMEM; }
        catch (const std::length_error &) { mine = CS_ENOMEM; }
        catch (...) { mine = CS_EINVAL; }
        if (mine != CS_OK) {
            int expect = CS_OK;
            rc.compare_exchange_strong(expect, mine);
            next.store(n);   // the others stop at their next index
        }
    };
    std::vector<std::thread> th;
    try {
        th.reserve(nt);
        for (int t = 1; t < nt; ++t) th.emplace_back(work);
    } catch (...) {}
    work();
    for (auto &t : th) t.join();
    return rc.load();
}

// Frees the cluster state of a context on every way out of cs_set_clusters but the successful one, exceptions included:
// a half-built state (maps and configurations listed, their device tables missing) must not survive the call.
struct ClustersGuard {
    cs_ctx *c;
    bool keep = false;
    ~ClustersGuard() { if (!keep) free_clusters(c); }
};

// Everything of one configuration that is computed on the host before anything is uploaded.
struct CfgPlanHost {
    SortedPlan sp;
    bool sorted = false;
    MapPlanHost mp[4];
    std::vector<int32_t> kp[4], kl[4];
    std::vector<int32_t> hdrptr;
    std::vector<uint32_t> hdrblob;
    std::vector<int32_t> live;   // [nregion]
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// TMA descriptor of d viewed as a 2-D fp32 tensor [ndata*2*nfreq rows, npix]; one box = all rows of one data set for
// 256 consecutive pixels (half a tile).  Only possible when rows are 16-byte aligned; otherwise the loader warp uses
// plain loads.
int make_tmap(cs_ctx *c, const float *d, int32_t ndata, CUtensorMap *tm, bool *have) {
    *have = false;
    std::memset(tm, 0, sizeof(*tm));
    if ((c->npix % 4) != 0 || (((uintptr_t)d) % 16) != 0) return CS_OK;
    static EncodeTiledFn enc = nullptr;
    if (!enc) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return CS_ECUDA;
        enc = (EncodeTiledFn)fn;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)c->npix, (cuuint64_t)ndata * 2 * c->nfreq};
    const cuuint64_t strides[1] = {(cuuint64_t)c->npix * 4};
    const cuuint32_t box[2] = {(cuuint32_t)HALF, (cuuint32_t)(2 * c->nfreq)}, es[2] = {1, 1};
    if (enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)d, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return CS_ECUDA;
    *have = true;
    return CS_OK;
}

// The dynamic shared memory limit is a per-device function attribute: set for every instantiation when a context is
// created on a device (a context is bound to the device current at cs_create).
template <int NF, int MODE>
cudaError_t configure_mode() {
    cudaError_t e = cudaFuncSetAttribute(k_like_direct<NF, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)direct_smem_bytes<NF>());
    if (e != cudaSuccess) return e;
    if (MODE != MODE_MAPS) e = cudaFuncSetAttribute(k_like_sc<NF, MODE == MODE_MAPS ? MODE_VALUE : MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sc_smem_bytes<NF>());
    return e;
}
template <int NF>
cudaError_t configure_nf() {
    cudaError_t e;
    if ((e = configure_mode<NF, MODE_VALUE>()) != cudaSuccess) return e;
    if ((e = configure_mode<NF, MODE_GRAD>()) != cudaSuccess) return e;
    if ((e = configure_mode<NF, MODE_MAPS>()) != cudaSuccess) return e;
    if ((e = configure_mode<NF, MODE_CMBVAR>()) != cudaSuccess) return e;
    return configure_mode<NF, MODE_CHI2>();
}

// Launches the fused kernels over nrun_sc sorted-cell runs followed by nrun_dir direct runs at `runs`.
template <int NF, int MODE>
int launch_like_t(cs_ctx *c, const LikeParams &P0, const Run *runs, int nrun_sc, int64_t W_sc, int nrun_dir, int64_t W_dir, cudaStream_t st) {
    const bool prof = c->prof_on && MODE == MODE_GRAD;
    for (int pass = 0; pass < 2; ++pass) {
        const int nrun = pass == 0 ? nrun_sc : nrun_dir;
        const int64_t W = pass == 0 ? W_sc : W_dir;
        if (nrun == 0 || W == 0) continue;
        LikeParams P = P0;
        P.runs = runs + (pass == 0 ? 0 : nrun_sc);
        P.nrun = nrun;
        P.W = W;
        const int grid = (int)std::min<int64_t>(W, c->nsm);
        if (prof) cudaEventRecord(c->prof_ev[2 * (c->prof_n % cs_ctx::PROF_RING)], st);
        if (pass == 0) {
            if (MODE == MODE_MAPS) return CS_EINVAL;
            k_like_sc<NF, MODE == MODE_MAPS ? MODE_VALUE : MODE><<<grid, SC_THREADS, sc_smem_bytes<NF>(), st>>>(P);
        } else {
            k_like_direct<NF, MODE><<<grid, DR_THREADS, direct_smem_bytes<NF>(), st>>>(c->tmap, P);
        }
        if (prof) { cudaEventRecord(c->prof_ev[2 * (c->prof_n % cs_ctx::PROF_RING) + 1], st); c->prof_n++; }
        c->launches++;
    }
    CK(cudaGetLastError());
    return CS_OK;
}

template <int MODE>
int launch_like(cs_ctx *c, const LikeParams &P, const Run *runs, int nrun_sc, int64_t W_sc, int nrun_dir, int64_t W_dir, cudaStream_t st) {
    if (c->nfreq == 15) return launch_like_t<15, MODE>(c, P, runs, nrun_sc, W_sc, nrun_dir, W_dir, st);
    return launch_like_t<16, MODE>(c, P, runs, nrun_sc, W_sc, nrun_dir, W_dir, st);
}
template <int MODE>
int launch_batch(cs_ctx *c, const LikeParams &P, cudaStream_t st) {
    return launch_like<MODE>(c, P, c->d_runs, c->nrun_sc, c->W_sc, c->nrun_dir, c->W_dir, st);
}

LikeParams base_params(cs_ctx *c) {
    LikeParams P;
    std::memset(&P, 0, sizeof(P));
    P.d = c->d;
    P.npix = c->npix;
    P.nfreq = c->nfreq;
    P.use_tma = c->have_tmap ? 1 : 0;
    const int64_t stream_bytes = std::max<int64_t>((int64_t)c->ndata * c->nfreq * 2 * c->npix * 4, c->copy_bytes);
    P.evict_first = (stream_bytes > (int64_t)96 << 20) ? 1 : 0;
    P.ring_maps = 0;
    P.dcopy = c->d_copy;
    P.pinfo = c->d_pinfo;
    P.maps = c->d_maps;
    P.cfgs = c->d_cfgs;
    P.elist = c->d_elist;
    P.skip = c->skip;
    P.tab = c->d_tab;
    P.partial = c->d_partial;
    P.PS = c->PS;
    P.maps_out = nullptr;
    P.err = c->d_err;
    P.pcopy = c->d_pcopy;
    for (int f = 0; f < NROW; ++f) {
        const double l2 = c->tc.lnd[f] * 1.4426950408889634074;   // log2(nu_f/nu0d); 0 beyond nfreq (cd = 0 there)
        P.cdf[f] = (float)c->tc.cd[f]; P.l2h[f] = (float)l2; P.l2l[f] = (float)(l2 - (double)P.l2h[f]);
    }
    P.kc = c->kc;
    return P;
}

int ready(cs_ctx *c) {
    if (!c || c->maps.empty() || !c->d || !c->have_ninv || c->batch <= 0) return CS_EINVAL;
    return CS_OK;
}

// Gathers the private copies [j0, j1) of the sorted layout from the caller's data (k_relayout).
int relayout(cs_ctx *c, const float *d, int64_t j0, int64_t j1, cudaStream_t st) {
    for (int64_t j = j0; j < j1; j += 65535) {
        const int nj = (int)std::min<int64_t>(65535, j1 - j);
        dim3 grid(c->job_ntile_max, nj);
        k_relayout<<<grid, TPX, 0, st>>>(d, c->npix, 2 * c->nfreq, c->d_cfgs, c->d_jobs + j, c->d_copy);
        c->launches++;
    }
    CK(cudaGetLastError());
    return CS_OK;
}

int set_data_impl(cs_ctx *c, int32_t ndata, const float *d, const float *ninv, bool do_relayout) {
    if (!c || ndata <= 0 || !d || !ninv) return CS_EINVAL;
    for (int e = 0; e < c->batch; ++e)   // validate against the current batch before anything is changed
        if (c->data_of[e] >= ndata) return CS_EINVAL;
    float w[NROW] = {0};
    CK(cudaMemcpy(w, ninv, sizeof(float) * c->nfreq, cudaMemcpyDefault));
    double m00 = 0;
    for (int f = 0; f < c->nfreq; ++f) {
        if (!(w[f] > 0.f) || !std::isfinite(w[f])) return CS_EINVAL;
        m00 += (double)w[f];
    }
    CUtensorMap tm;
    bool have = false;
    int rc = make_tmap(c, d, ndata, &tm, &have);
    if (rc) return rc;
    std::memset(&c->kc, 0, sizeof(c->kc));
    for (int f = 0; f < c->nfreq; ++f) {
        c->kc.w[f] = w[f];
        c->kc.lnd[f] = (float)c->tc.lnd[f];
        c->kc.lns[f] = (float)c->tc.lns[f];
        c->kc.invw[f] = 1.0f / w[f];
    }
    c->kc.m00 = (float)m00;
    c->kc.inv_m00 = (float)(1.0 / m00);
    c->d = d;
    c->ndata = ndata;
    c->have_ninv = true;
    c->have_moments = false;   // f3 moments belong to the previous data
    c->tmap = tm;
    c->have_tmap = have;
    if (do_relayout && c->batch > 0 && !c->jobs.empty()) {
        if ((rc = relayout(c, d, 0, (int64_t)c->jobs.size(), nullptr))) return rc;
        CK(cudaDeviceSynchronize());
    }
    return CS_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------
extern "C" {

int cs_version(void) { return 2; }

const char *cs_strerror(int code) {
    switch (code) {
        case CS_OK: return "ok";
        case CS_EINVAL: return "invalid argument or call order";
        case CS_EINDEX: return "cluster or region index out of range";
        case CS_EDOMAIN: return "T_d <= 0 or non-finite spectral parameter";
        case CS_ESINGULAR: return "singular A^T N^-1 A";
        case CS_ECUDA: return "CUDA runtime error";
        case CS_ENOMEM: return "out of device memory";
        case CS_ELIMIT: return "size beyond the fixed capacity of a no-allocation entry point";
        default: return "unknown error";
    }
}

int cs_create(cs_ctx **out, const cs_model *m) {
    if (!out) return CS_EINVAL;
    *out = nullptr;
    if (!m || !m->freqs_ghz || m->nfreq < 3 || m->nfreq > CS_MAX_NFREQ || m->npix <= 0 || m->npix > (int64_t)0x7fff0000)
        return CS_EINVAL;
    if (!(m->nu0_dust_ghz > 0) || !(m->nu0_sync_ghz > 0) || !(m->t_cmb_k > 0)) return CS_EINVAL;
    if (m->units != CS_UNITS_KCMB && m->units != CS_UNITS_LITERAL) return CS_EINVAL;
    for (int f = 0; f < m->nfreq; ++f)
        if (!(m->freqs_ghz[f] > 0) || !std::isfinite(m->freqs_ghz[f])) return CS_EINVAL;
    cs_ctx *c = new (std::nothrow) cs_ctx();
    if (!c) return CS_ENOMEM;
    c->nfreq = m->nfreq; c->units = m->units; c->npix = m->npix;
    c->ntile_ring = (int32_t)((m->npix + TPX - 1) / TPX);
    c->nu0d = m->nu0_dust_ghz; c->nu0s = m->nu0_sync_ghz; c->tcmb = m->t_cmb_k;
    // exact SI constants (R3)
    const double hk = 6.62607015e-34 * 1e9 / 1.380649e-23;
    std::memset(&c->tc, 0, sizeof(c->tc));
    std::memset(&c->kc, 0, sizeof(c->kc));
    c->tc.nfreq = m->nfreq; c->tc.nu0d = c->nu0d; c->tc.hk = hk;
    const double u0d = krj2kcmb(c->nu0d, c->tcmb, hk), u0s = krj2kcmb(c->nu0s, c->tcmb, hk);
    for (int f = 0; f < m->nfreq; ++f) {
        const double nu = m->freqs_ghz[f];
        c->freqs[f] = nu;
        const double ud = m->units == CS_UNITS_KCMB ? krj2kcmb(nu, c->tcmb, hk) / u0d : 1.0;
        const double us = m->units == CS_UNITS_KCMB ? krj2kcmb(nu, c->tcmb, hk) / u0s : 1.0;
        c->tc.nu[f] = nu;
        c->tc.lnd[f] = std::log(nu / c->nu0d);
        c->tc.lns[f] = std::log(nu / c->nu0s);
        c->tc.cd[f] = (nu / c->nu0d) * ud;   // (nu/nu0)^(beta_d+1) = (nu/nu0) * (nu/nu0)^beta_d
        c->tc.cs[f] = us;
    }
    int dev = 0, nsm = 0;
    bool ok = cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0;
    ok = ok && configure_nf<15>() == cudaSuccess && configure_nf<16>() == cudaSuccess;
    ok = ok && cudaMalloc((void **)&c->d_err, sizeof(int32_t)) == cudaSuccess && cudaMemset(c->d_err, 0, sizeof(int32_t)) == cudaSuccess &&
         cudaMalloc((void **)&c->d_tc, sizeof(TConst)) == cudaSuccess &&
         cudaMemcpy(c->d_tc, &c->tc, sizeof(TConst), cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) {
        cudaFree(c->d_err); cudaFree(c->d_tc);
        delete c;
        return CS_ECUDA;
    }
    c->nsm = nsm;
    *out = c;
    return CS_OK;
}

int cs_destroy(cs_ctx *c) {
    if (!c) return CS_EINVAL;
    cudaDeviceSynchronize();
    free_batch(c);
    free_clusters(c);
    cudaFree(c->d_stage);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->comp_stream) cudaStreamDestroy(c->comp_stream);
    cudaFree(c->d_err);
    cudaFree(c->d_tc);
    for (auto &e : c->prof_ev) cudaEventDestroy(e);
    for (auto &e : c->sel_ev) if (e) cudaEventDestroy(e);
    delete c;
    return CS_OK;
}

int cs_model_constants(cs_ctx *c, double *cd, double *cs_, double *lnd, double *lns, double *inv_sum_w) {
    if (!c) return CS_EINVAL;
    for (int f = 0; f < c->nfreq; ++f) {
        if (cd) cd[f] = c->tc.cd[f];
        if (cs_) cs_[f] = c->tc.cs[f];
        if (lnd) lnd[f] = c->tc.lnd[f];
        if (lns) lns[f] = c->tc.lns[f];
    }
    if (inv_sum_w) *inv_sum_w = c->have_ninv ? (double)c->kc.inv_m00 : 0.0;
    return CS_OK;
}

int cs_set_option(cs_ctx *c, int32_t key, double value) {
    if (!c || !std::isfinite(value)) return CS_EINVAL;
    switch (key) {
        case CS_OPT_LAYOUT:
            if (value != CS_LAYOUT_AUTO && value != CS_LAYOUT_INPLACE && value != CS_LAYOUT_SORTED) return CS_EINVAL;
            if (!c->maps.empty()) return CS_EINVAL;   // decided when the clusters are set
            c->opt_layout = (int32_t)value;
            return CS_OK;
        case CS_OPT_FORM:
            if (value != CS_FORM_AUTO && value != CS_FORM_DIRECT) return CS_EINVAL;
            if (c->batch > 0) return CS_EINVAL;       // decided when the batch is set
            c->opt_form = (int32_t)value;
            return CS_OK;
        case CS_OPT_MIN_FILL:
            if (!(value >= 0.0 && value <= 1.0) || !c->maps.empty()) return CS_EINVAL;
            c->opt_min_fill = value;
            return CS_OK;
        case CS_OPT_PIXEL_BETA:
            if (value != CS_PIXBETA_AUTO && value != CS_PIXBETA_OFF) return CS_EINVAL;
            if (!c->maps.empty()) return CS_EINVAL;   // decided when the clusters are set
            c->opt_pixbeta = (int32_t)value;
            return CS_OK;
        case CS_OPT_COPY_LIMIT_MB:
            if (value < 0) return CS_EINVAL;
            c->opt_copy_limit = (int64_t)(value * 1048576.0);
            return CS_OK;
        default:
            return CS_EINVAL;
    }
}

int cs_set_clusters(cs_ctx *c, int32_t nmap, const int32_t *maps, const int32_t *Kmap, int32_t ncfg,
                    const int32_t *cfg_maps, const uint8_t *region_idx, int32_t nregion) {
    if (!c || nmap <= 0 || !maps || !Kmap || ncfg <= 0 || !cfg_maps || nregion < 1 || nregion > 255) return CS_EINVAL;
    if (nregion > 1 && !region_idx) return CS_EINVAL;
    CS_GUARD_BEGIN
    const int64_t npix = c->npix;
    for (int32_t m = 0; m < nmap; ++m)
        if (Kmap[m] <= 0) return CS_EINVAL;
    for (int32_t i = 0; i < ncfg * 3; ++i)
        if (cfg_maps[i] < 0 || cfg_maps[i] >= nmap) return CS_EINVAL;
    // bring the maps to the host (plan building is a once-per-clustering step, not on the hot path)
    std::vector<int32_t> h((size_t)nmap * npix);
    CK(cudaMemcpy(h.data(), maps, h.size() * sizeof(int32_t), cudaMemcpyDefault));
    std::vector<int32_t> reg(npix, 0);
    if (region_idx) {
        std::vector<uint8_t> r8(npix);
        CK(cudaMemcpy(r8.data(), region_idx, (size_t)npix, cudaMemcpyDefault));
        for (int64_t p = 0; p < npix; ++p) {
            if (r8[p] >= nregion) return CS_EINDEX;
            reg[p] = r8[p];
        }
    }
    // bit-exact index validation before anything is changed
    for (int32_t m = 0; m < nmap; ++m) {
        const int32_t *ix = h.data() + (size_t)m * npix;
        const int32_t K = Kmap[m];
        for (int64_t p = 0; p < npix; ++p)
            if (ix[p] < -1 || ix[p] >= K) return CS_EINDEX;
    }
    cudaDeviceSynchronize();
    free_batch(c);
    free_clusters(c);
    ClustersGuard guard{c};
    c->maps.resize(nmap + 1);
    int rc;
    {   // pixel-space plans of the nmap cluster maps and of the region pseudo-map
        std::vector<MapPlanHost> pm(nmap + 1);
        if ((rc = parallel_for(nmap + 1, [&](int m) {
                if (m < nmap) compute_map_plan(h.data() + (size_t)m * npix, Kmap[m], npix, c->ntile_ring, pm[m]);
                else compute_map_plan(reg.data(), nregion, npix, c->ntile_ring, pm[m]);
            }))) return rc;
        for (int32_t m = 0; m <= nmap; ++m)
            if ((rc = upload_map_plan(c->cl_arena, pm[m], &c->maps[m], &c->cluster_bytes))) { free_clusters(c); return rc; }
    }
    c->nmap = nmap; c->ncfg = ncfg; c->nregion = nregion;
    c->cfgs.resize(ncfg);
    c->sorted.resize(ncfg);
    c->cellsh.resize(ncfg);
    c->npix_live.assign((size_t)ncfg * nregion, 0);
    for (int32_t i = 0; i < ncfg; ++i) {
        CfgDev &cf = c->cfgs[i];
        std::memset(&cf, 0, sizeof(cf));
        for (int t = 0; t < 4; ++t) {
            cf.rmap[t] = t < 3 ? cfg_maps[i * 3 + t] : nmap;
            cf.map[t] = cf.rmap[t];
            if (t < 3) cf.K[t] = Kmap[cf.rmap[t]];
        }
        cf.ktot = cf.K[0] + cf.K[1] + cf.K[2];
        cf.ntile = cf.ntile_ring = c->ntile_ring;
    }
    // configurations in groups: the host part of a group on all threads (sorted layout, the four position-space plans,
    // the cell lists, the tile headers), then its uploads in order
    constexpr int GROUP = 32;
    std::vector<CfgPlanHost> plans(std::min<int32_t>(GROUP, ncfg));
    for (int32_t i0 = 0; i0 < ncfg; i0 += GROUP) {
        const int32_t ng = std::min<int32_t>(GROUP, ncfg - i0);
        if ((rc = parallel_for(ng, [&](int g) {
                const int32_t i = i0 + g;
                const CfgDev &cf = c->cfgs[i];
                CfgPlanHost &pl = plans[g];
                const int32_t *a = h.data() + (size_t)cf.rmap[0] * npix, *b = h.data() + (size_t)cf.rmap[1] * npix,
                              *d = h.data() + (size_t)cf.rmap[2] * npix;
                pl.live.assign(nregion, 0);
                for (int64_t p = 0; p < npix; ++p)
                    if (a[p] >= 0 && b[p] >= 0 && d[p] >= 0) pl.live[reg[p]]++;
                pl.sorted = false;
                // sorted layout: taken when the option asks for it, or (auto) when its tiles come out well filled --
                // small cells (K ~ npix) would mostly stream padding
                if (c->opt_layout == CS_LAYOUT_INPLACE) return;
                plan_sorted(a, b, d, reg.data(), cf.K, npix, pl.sp);
                if (!(c->opt_layout == CS_LAYOUT_SORTED || pl.sp.fill >= c->opt_min_fill)) return;
                pl.sorted = true;
                const int64_t npos = (int64_t)pl.sp.ntile * TPX;
                int32_t segbase[4], off = 0;
                for (int t = 0; t < 4; ++t) {
                    compute_map_plan(pl.sp.idx[t].data(), t < 3 ? cf.K[t] : nregion, npos, pl.sp.ntile, pl.mp[t]);
                    segbase[t] = off;
                    off += pl.mp[t].nseg;
                }
                const int32_t ncell = (int32_t)pl.sp.cellpos.size();   // global cell list (f3): cluster / region -> cells
                for (int t = 0; t < 4; ++t) {
                    const int32_t Kt = t < 3 ? cf.K[t] : nregion;
                    std::vector<int32_t> &kp = pl.kp[t], &kl = pl.kl[t];
                    kp.assign(Kt + 1, 0); kl.assign(ncell, 0);
                    for (int32_t q = 0; q < ncell; ++q) kp[pl.sp.cellkey[t][q] + 1]++;
                    for (int32_t k = 0; k < Kt; ++k) kp[k + 1] += kp[k];
                    std::vector<int32_t> fill(kp.begin(), kp.end() - 1);
                    for (int32_t q = 0; q < ncell; ++q) kl[fill[pl.sp.cellkey[t][q]]++] = q;
                }
                pack_tile_headers(pl.sp, pl.mp, segbase, pl.mp[3].nseg, pl.hdrptr, pl.hdrblob);   // they hold the slots
            }))) return rc;
        for (int32_t g = 0; g < ng; ++g) {
            const int32_t i = i0 + g;
            CfgDev &cf = c->cfgs[i];
            CfgPlanHost &pl = plans[g];
            for (int32_t r = 0; r < nregion; ++r) c->npix_live[(size_t)i * nregion + r] = pl.live[r];
            if (pl.sorted) {
                const SortedPlan &sp = pl.sp;
                SortedHost &sh = c->sorted[i];
                CellsHost &ch = c->cellsh[i];
                ch.ncell = (int32_t)sp.cellpos.size();
                c->ncell_max = std::max(c->ncell_max, ch.ncell);
                if ((rc = arena_upload(c->cl_arena, &sh.cellid, sp.cellid, &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &sh.cellptr, sp.cellptr, &c->cluster_bytes)) ||
                    (rc = arena_upload(c->cl_arena, &sh.cellrows, sp.cellrows, &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &sh.pospix, sp.pospix, &c->cluster_bytes)) ||
                    (rc = arena_upload(c->cl_arena, &ch.cellpos, sp.cellpos, &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &ch.celllen, sp.celllen, &c->cluster_bytes)) ||
                    (rc = arena_upload(c->cl_arena, &ch.cellreg, sp.cellkey[3], &c->cluster_bytes)) ||
                    (rc = arena_upload(c->cl_arena, &sh.hdr, pl.hdrblob, &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &sh.hdrptr, pl.hdrptr, &c->cluster_bytes))) {
                    free_clusters(c);
                    return rc;
                }
                for (int t = 0; t < 4; ++t) {
                    c->maps.emplace_back();
                    if ((rc = upload_map_plan(c->cl_arena, pl.mp[t], &c->maps.back(), &c->cluster_bytes)) ||
                        (rc = arena_upload(c->cl_arena, &ch.kptr[t], pl.kp[t], &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &ch.klist[t], pl.kl[t], &c->cluster_bytes))) {
                        free_clusters(c);
                        return rc;
                    }
                    cf.map[t] = (int32_t)c->maps.size() - 1;
                }
                cf.sorted = 1;
                cf.ntile = sp.ntile;
                cf.cellid = sh.cellid; cf.cellptr = sh.cellptr; cf.cellrows = sh.cellrows; cf.pospix = sh.pospix;
                cf.hdr = sh.hdr; cf.hdrptr = sh.hdrptr;
            }
            cf.pixbeta = (!cf.sorted && c->opt_pixbeta == CS_PIXBETA_AUTO && 2 * (int64_t)cf.K[0] > npix) ? 1 : 0;
            int32_t off = 0;
            for (int t = 0; t < 4; ++t) {
                cf.segbase[t] = off;
                cf.kseg[t] = c->maps[cf.map[t]].ksegptr;
                off += c->maps[cf.map[t]].nseg;
            }
        }
    }
    std::vector<MapDev> md(c->maps.size());
    for (size_t m = 0; m < c->maps.size(); ++m) {
        const MapHost &s = c->maps[m];
        md[m] = MapDev{s.idx, s.rank, s.segptr, s.segdesc, s.segslot, s.ksegptr, s.chunkptr, s.segcfirst, s.K, s.nseg};
    }
    std::vector<CellsDev> cd(ncfg);
    for (int32_t i = 0; i < ncfg; ++i) {
        const CellsHost &ch = c->cellsh[i];
        std::memset(&cd[i], 0, sizeof(CellsDev));
        cd[i].cellpos = ch.cellpos; cd[i].celllen = ch.celllen; cd[i].cellrows = c->sorted[i].cellrows; cd[i].cellreg = ch.cellreg;
        for (int t = 0; t < 4; ++t) { cd[i].kptr[t] = ch.kptr[t]; cd[i].klist[t] = ch.klist[t]; }
        cd[i].ncell = ch.ncell;
    }
    if ((rc = arena_upload(c->cl_arena, &c->d_maps, md, &c->cluster_bytes)) || (rc = arena_upload(c->cl_arena, &c->d_cfgs, c->cfgs, &c->cluster_bytes)) ||
        (rc = arena_upload(c->cl_arena, &c->d_cells, cd, &c->cluster_bytes)) ||
        (rc = arena_upload(c->cl_arena, &c->d_npix_live, c->npix_live, &c->cluster_bytes)))
        return rc;
    guard.keep = true;
    return CS_OK;
    CS_GUARD_END
}

int cs_layout_info(cs_ctx *c, int32_t cfg, int32_t *sorted, int32_t *ntile, double *fill) {
    if (!c || cfg < 0 || cfg >= c->ncfg) return CS_EINVAL;
    const CfgDev &cf = c->cfgs[cfg];
    int64_t live = 0;
    for (int r = 0; r < c->nregion; ++r) live += c->npix_live[(size_t)cfg * c->nregion + r];
    if (sorted) *sorted = cf.sorted;
    if (ntile) *ntile = cf.ntile;
    if (fill) *fill = (double)live / ((double)cf.ntile * TPX);
    return CS_OK;
}

int cs_set_data(cs_ctx *c, int32_t ndata, const float *d, const float *ninv) { return set_data_impl(c, ndata, d, ninv, true); }

int cs_set_batch(cs_ctx *c, int32_t batch, const int32_t *cfg_of, const int32_t *data_of) {
    if (!c || c->maps.empty() || batch <= 0 || !cfg_of || !data_of) return CS_EINVAL;
    for (int32_t e = 0; e < batch; ++e) {
        if (cfg_of[e] < 0 || cfg_of[e] >= c->ncfg || data_of[e] < 0) return CS_EINVAL;
        if (c->d && data_of[e] >= c->ndata) return CS_EINVAL;
    }
    CS_GUARD_BEGIN
    cudaDeviceSynchronize();
    free_batch(c);
    c->cfg_of.assign(cfg_of, cfg_of + batch);
    c->data_of.assign(data_of, data_of + batch);
    c->param_off.assign(batch + 1, 0);
    std::vector<int64_t> &tab_off = c->tab_off;
    tab_off.assign(batch, 0);
    const int32_t nseg_reg = c->maps[c->nmap].nseg;
    int64_t rows = 0, PS = 4 * (int64_t)nseg_reg;
    int32_t kmax = 0;
    for (int32_t e = 0; e < batch; ++e) {
        const CfgDev &cf = c->cfgs[cfg_of[e]];
        c->param_off[e + 1] = c->param_off[e] + cf.ktot;
        tab_off[e] = rows;
        rows += cf.K[0] + 2 * (int64_t)cf.K[1] + cf.K[2];
        const int64_t nreg = c->maps[cf.map[3]].nseg;
        PS = std::max<int64_t>(PS, std::max<int64_t>((int64_t)cf.segbase[3] + nreg, 4 * nreg));
        kmax = std::max(kmax, cf.ktot);
    }
    c->nparam = c->param_off[batch];
    c->nrows = rows; c->PS = PS; c->ktot_max = kmax;
    // entries ordered by (kernel form, configuration), stable; a run = all entries of one configuration
    const bool force_direct = c->opt_form == CS_FORM_DIRECT;
    c->elist.resize(batch);
    for (int32_t e = 0; e < batch; ++e) c->elist[e] = e;
    auto is_sc = [&](int32_t e) { return c->cfgs[cfg_of[e]].sorted && !force_direct; };
    auto key = [&](int32_t e) { return ((int64_t)(is_sc(e) ? 0 : 1) << 32) | (int64_t)cfg_of[e]; };
    std::stable_sort(c->elist.begin(), c->elist.end(), [&](int32_t a, int32_t b) { return key(a) < key(b); });
    c->runs.clear();
    c->nrun_sc = c->nrun_dir = 0;
    c->W_sc = c->W_dir = 0;
    for (int32_t i = 0; i < batch;) {
        int32_t j = i;
        while (j < batch && cfg_of[c->elist[j]] == cfg_of[c->elist[i]]) ++j;
        const CfgDev &cf = c->cfgs[cfg_of[c->elist[i]]];
        const bool sc = is_sc(c->elist[i]);
        Run r{cfg_of[c->elist[i]], i, j - i, cf.ntile, sc ? c->W_sc : c->W_dir, cf.hdr, cf.hdrptr, 0};   // tstride: below
        const int64_t units = (int64_t)cf.ntile * (j - i);
        if (sc) { c->W_sc += units; c->nrun_sc++; } else { c->W_dir += units; c->nrun_dir++; }
        c->runs.push_back(r);
        i = j;
    }
    // private copies of the sorted layout: one per (configuration, data set) pair, ordered by data set
    c->jobs.clear();
    c->cfg_tstride.assign(c->ncfg, 0);
    c->copy_off.assign(batch, -1);
    c->job_ntile_max = 0;
    int64_t copy_floats = 0;
    {
        std::map<std::pair<int32_t, int32_t>, int64_t> seen;   // (data, cfg) -> offset
        std::vector<std::pair<int32_t, int32_t>> order;
        for (int32_t e = 0; e < batch; ++e)
            if (c->cfgs[cfg_of[e]].sorted) {
                const auto k = std::make_pair(data_of[e], cfg_of[e]);
                if (seen.emplace(k, 0).second) order.push_back(k);
            }
        std::sort(order.begin(), order.end());
        // tile-major (cs_internal.h): the pairs of a configuration are interleaved tile by tile
        const int64_t blk = (int64_t)2 * c->nfreq * TPX;   // floats of one tile of one copy
        std::vector<int32_t> npair(c->ncfg, 0), pidx(order.size(), 0);
        for (size_t j = 0; j < order.size(); ++j) pidx[j] = npair[order[j].second]++;
        std::vector<int64_t> cfgbase(c->ncfg, 0);
        for (int32_t q = 0; q < c->ncfg; ++q) {
            cfgbase[q] = copy_floats;
            copy_floats += (int64_t)c->cfgs[q].ntile * npair[q] * blk * (npair[q] > 0 ? 1 : 0);
            c->cfg_tstride[q] = (int64_t)npair[q] * blk;
        }
        for (size_t j = 0; j < order.size(); ++j) {
            const auto &k = order[j];
            const CfgDev &cf = c->cfgs[k.second];
            const int64_t off = cfgbase[k.second] + (int64_t)pidx[j] * blk;
            seen[k] = off;
            c->jobs.push_back(CopyJob{k.second, k.first, off, c->cfg_tstride[k.second]});
            c->job_ntile_max = std::max(c->job_ntile_max, cf.ntile);
        }
        for (int32_t e = 0; e < batch; ++e)
            if (c->cfgs[cfg_of[e]].sorted) c->copy_off[e] = seen[std::make_pair(data_of[e], cfg_of[e])];
    }
    for (Run &r : c->runs) r.tstride = c->cfg_tstride[r.cfg];
    c->pinfo.resize(batch);
    for (int32_t i = 0; i < batch; ++i) {
        const int32_t e = c->elist[i];
        c->pinfo[i] = PosInfo{tab_off[e], c->cfgs[cfg_of[e]].sorted ? c->copy_off[e] : (int64_t)data_of[e], c->param_off[e], 0};
    }
    const int64_t copy_bytes = copy_floats * 4;
    if (copy_bytes > 0) {
        int64_t limit = c->opt_copy_limit;
        if (limit == 0) {
            size_t fr = 0, tot = 0;
            CK(cudaMemGetInfo(&fr, &tot));
            limit = (int64_t)(0.7 * (double)fr);
        }
        if (copy_bytes > limit) { free_batch(c); return CS_ENOMEM; }
    }
    std::vector<TabBlock> tabblk;
    c->any_pixbeta = false;
    for (int32_t e = 0; e < batch; ++e) {
        const CfgDev &cf = c->cfgs[cfg_of[e]];
        c->any_pixbeta = c->any_pixbeta || cf.pixbeta != 0;
        for (int32_t j0 = 0; j0 < cf.ktot; j0 += TAB_ROWS_PER_BLOCK)
            // (a block that lies wholly in the beta_d rows of a pixbeta configuration builds nothing, but still checks
            // its parameters: CS_EDOMAIN is raised here, whichever kernel evaluates the power law)
            tabblk.push_back(TabBlock{c->param_off[e], tab_off[e], cf.K[0], cf.K[1], cf.ktot, j0, e, cf.pixbeta, {0, 0}});
    }
    c->ntabblk = (int64_t)tabblk.size();
    std::vector<MergeBlock> mblk;
    for (int32_t e = 0; e < batch; ++e)
        for (int32_t r = 0; r < c->nregion; ++r) mblk.push_back(MergeBlock{e, -(r + 1)});
    c->nmblk_region = (int64_t)mblk.size();
    for (int32_t e = 0; e < batch; ++e)
        for (int32_t b = 0; b * 256 < c->cfgs[cfg_of[e]].ktot; ++b) mblk.push_back(MergeBlock{e, b});
    c->nmblk_all = (int64_t)mblk.size();
    int rc;
    if ((rc = dev_upload(&c->d_tabblk, tabblk, &c->batch_bytes)) || (rc = dev_upload(&c->d_mblk, mblk, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_cfg_of, c->cfg_of, &c->batch_bytes)) || (rc = dev_upload(&c->d_data_of, c->data_of, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_elist, c->elist, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_param_off, c->param_off, &c->batch_bytes)) || (rc = dev_upload(&c->d_tab_off, tab_off, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_pinfo, c->pinfo, &c->batch_bytes)) || (rc = dev_upload(&c->d_runs, c->runs, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_jobs, c->jobs, &c->batch_bytes))) {
        free_batch(c);
        return rc;
    }
    const size_t tab_bytes = (size_t)rows * NROW * sizeof(float), part_bytes = (size_t)batch * PS * sizeof(double);
    c->sel_cap = (((int64_t)batch * (1 + (int64_t)((sizeof(Run) + sizeof(PosInfo)) / 4)) + 16) + 3) & ~(int64_t)3;   // slots stay 16-byte aligned
    if (cudaMalloc((void **)&c->d_tab, tab_bytes) != cudaSuccess || cudaMalloc((void **)&c->d_partial, part_bytes) != cudaSuccess ||
        cudaMalloc((void **)&c->d_pcopy, (size_t)std::max<int64_t>(c->nparam, 1) * sizeof(double)) != cudaSuccess ||
        (copy_bytes > 0 && cudaMalloc((void **)&c->d_copy, (size_t)copy_bytes) != cudaSuccess) ||
        cudaMalloc((void **)&c->d_sel, (size_t)(cs_ctx::SEL_RING * c->sel_cap * 4)) != cudaSuccess ||
        cudaMallocHost((void **)&c->h_sel, (size_t)(cs_ctx::SEL_RING * c->sel_cap * 4)) != cudaSuccess) {
        cudaGetLastError();
        free_batch(c);
        return CS_ENOMEM;
    }
    c->batch_bytes += (int64_t)(tab_bytes + part_bytes) + c->nparam * 8 + copy_bytes + cs_ctx::SEL_RING * c->sel_cap * 4;
    c->copy_bytes = copy_bytes;
    c->batch = batch;
    if (c->d && !c->jobs.empty()) {
        if ((rc = relayout(c, c->d, 0, (int64_t)c->jobs.size(), nullptr))) { free_batch(c); return rc; }
        CK(cudaDeviceSynchronize());
    }
    return CS_OK;
    CS_GUARD_END
}

int cs_param_offsets(cs_ctx *c, int64_t *off) {
    if (!c || c->batch <= 0 || !off) return CS_EINVAL;
    std::memcpy(off, c->param_off.data(), sizeof(int64_t) * (c->batch + 1));
    return CS_OK;
}

int cs_build_sed_tables(cs_ctx *c, const double *params, void *stream) {
    if (!c || c->batch <= 0 || !params) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // the parameters the tables belong to: read only by the per-pixel beta_d path of the direct kernel
    if (c->any_pixbeta) CK(cudaMemcpyAsync(c->d_pcopy, params, (size_t)c->nparam * sizeof(double), cudaMemcpyDeviceToDevice, st));
    if (c->ntabblk > 0)
        k_tables<<<(unsigned)c->ntabblk, 256, 0, st>>>(params, c->d_tabblk, c->d_tab, c->d_err, c->d_tc, c->skip);
    c->launches++;
    CK(cudaGetLastError());
    c->tables_built = true;
    return CS_OK;
}

static int merge_launch(cs_ctx *c, double *nll, double *grad, cudaStream_t st) {
    const int64_t nblk = grad ? c->nmblk_all : c->nmblk_region;   // value only: the region blocks at the head of the list
    if (nblk > 0) {
        k_merge<<<(unsigned)nblk, 256, 0, st>>>(c->d_partial, c->PS, c->d_cfgs, c->d_cfg_of, c->d_param_off, c->nregion, c->d_mblk, nll, grad, c->skip);
        c->launches++;
    }
    CK(cudaGetLastError());
    return CS_OK;
}

int cs_spectral_like_grad(cs_ctx *c, double *nll, double *grad, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!nll || !c->tables_built) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LikeParams P = base_params(c);
    rc = grad ? launch_batch<MODE_GRAD>(c, P, st) : launch_batch<MODE_VALUE>(c, P, st);
    if (rc) return rc;
    return merge_launch(c, nll, grad, st);
}

int cs_spectral_misfit(cs_ctx *c, double *chi2, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!chi2 || !c->tables_built) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LikeParams P = base_params(c);
    if ((rc = launch_batch<MODE_CHI2>(c, P, st))) return rc;
    return merge_launch(c, chi2, nullptr, st);
}

// a4 and the map level of f4(ii): W(params of entry e) applied to data set data_sel[i] (or the entry's own), `planes`
// output planes per selected entry.
static int maps_impl(cs_ctx *c, int32_t nsel, const int32_t *entries, const int32_t *data_sel, int32_t planes, float *s, cudaStream_t st) {
    int rc = ready(c);
    if (rc) return rc;
    if (!s || !c->tables_built || nsel <= 0 || nsel > c->batch) return CS_EINVAL;
    if (!entries && nsel != c->batch) return CS_EINVAL;
    // The selection (entry list, per-position info, then its runs = stretches of consecutive selected entries of one
    // configuration) goes through a small ring of pinned staging slots, so that the call never synchronises the
    // caller's stream; a slot (host and device side) is reused only after the kernel that read it has completed.
    const int slot = (int)(c->sel_n % cs_ctx::SEL_RING);
    if (!c->sel_ev[slot]) CK(cudaEventCreateWithFlags(&c->sel_ev[slot], cudaEventDisableTiming));
    else CK(cudaEventSynchronize(c->sel_ev[slot]));
    int32_t *hs = c->h_sel + slot * c->sel_cap, *ds = c->d_sel + slot * c->sel_cap;
    for (int32_t i = 0; i < nsel; ++i) {
        const int32_t e = entries ? entries[i] : i;
        if (e < 0 || e >= c->batch) return CS_EINVAL;
        if (data_sel && (data_sel[i] < 0 || data_sel[i] >= c->ndata)) return CS_EINVAL;
        hs[i] = e;
    }
    const int64_t poff = ((int64_t)nsel + 3) & ~(int64_t)3;   // position info starts 16-byte aligned, the runs follow it
    PosInfo *hp = reinterpret_cast<PosInfo *>(hs + poff);
    for (int32_t i = 0; i < nsel; ++i) hp[i] = PosInfo{c->tab_off[hs[i]], (int64_t)(data_sel ? data_sel[i] : c->data_of[hs[i]]), c->param_off[hs[i]], 0};
    const int64_t roff = poff + (int64_t)nsel * (int64_t)(sizeof(PosInfo) / 4);
    Run *hr = reinterpret_cast<Run *>(hs + roff);
    int32_t nrun = 0;
    int64_t W = 0;
    for (int32_t i = 0; i < nsel;) {
        const int32_t cf = c->cfg_of[hs[i]];
        int32_t j = i;
        while (j < nsel && c->cfg_of[hs[j]] == cf) ++j;
        hr[nrun++] = Run{cf, i, j - i, c->ntile_ring, W, nullptr, nullptr, 0};
        W += (int64_t)c->ntile_ring * (j - i);
        i = j;
    }
    const size_t bytes = (size_t)roff * 4 + (size_t)nrun * sizeof(Run);
    CK(cudaMemcpyAsync(ds, hs, bytes, cudaMemcpyHostToDevice, st));
    c->sel_n++;
    LikeParams P = base_params(c);
    P.elist = ds;
    P.pinfo = reinterpret_cast<const PosInfo *>(ds + poff);
    P.maps_out = s;
    P.maps_planes = planes;
    P.ring_maps = 1;
    P.evict_first = ((int64_t)c->ndata * c->nfreq * 2 * c->npix * 4 > (int64_t)96 << 20) ? 1 : 0;
    rc = launch_like<MODE_MAPS>(c, P, reinterpret_cast<const Run *>(ds + roff), 0, 0, nrun, W, st);
    // after the launch, not after the copy: the kernel reads the device side of the slot, whichever stream it ran on
    const cudaError_t ev = cudaEventRecord(c->sel_ev[slot], st);
    return rc ? rc : (ev == cudaSuccess ? CS_OK : CS_ECUDA);
}

int cs_component_maps(cs_ctx *c, int32_t nsel, const int32_t *entries, float *s, void *stream) {
    return maps_impl(c, nsel, entries, nullptr, 6, s, (cudaStream_t)stream);
}

int cs_cmb_residual_maps(cs_ctx *c, int32_t nsel, const int32_t *entries, const int32_t *data_sel, float *cmb, void *stream) {
    if (!data_sel) return CS_EINVAL;
    return maps_impl(c, nsel, entries, data_sel, 2, cmb, (cudaStream_t)stream);
}

int cs_cell_moments(cs_ctx *c, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (c->nfreq > CC_MAXF) return CS_EINVAL;
    for (int32_t e = 0; e < c->batch; ++e)
        if (!c->cfgs[c->cfg_of[e]].sorted) return CS_EINVAL;   // f3 needs the cell list of the sorted layout
    CS_GUARD_BEGIN
    cudaStream_t st = (cudaStream_t)stream;
    if (!c->d_mom) {   // workspace: moments of every (configuration, data set) pair, per-cell terms, offsets
        std::vector<MomJob> mj(c->jobs.size());
        std::map<std::pair<int32_t, int32_t>, int64_t> off;
        int64_t n = 0;
        for (size_t j = 0; j < c->jobs.size(); ++j) {
            mj[j] = MomJob{c->jobs[j].cfg, c->jobs[j].data, n, c->jobs[j].off, c->jobs[j].tstride};
            off[std::make_pair(c->jobs[j].data, c->jobs[j].cfg)] = n;
            n += (int64_t)CC_NMOM * c->cellsh[c->jobs[j].cfg].ncell;
        }
        std::vector<int64_t> mo(c->batch);
        for (int32_t e = 0; e < c->batch; ++e) mo[e] = off[std::make_pair(c->data_of[e], c->cfg_of[e])];
        c->cc_out_stride = 4 * (int64_t)((c->ncell_max + 31) & ~31);
        const size_t out_bytes = (size_t)c->batch * c->cc_out_stride * sizeof(double);
        int64_t b = 0;
        // all five buffers or none: d_mom != nullptr is what marks the workspace as present on the next call
        auto drop = [&]() {
            cudaFree(c->d_mom); cudaFree(c->d_ccout); cudaFree(c->d_mom_off); cudaFree(c->d_momjobs); cudaFree(c->d_w);
            c->d_mom = c->d_ccout = nullptr; c->d_mom_off = nullptr; c->d_momjobs = nullptr; c->d_w = nullptr;
            cudaGetLastError();
        };
        if ((rc = dev_upload(&c->d_momjobs, mj, &b)) || (rc = dev_upload(&c->d_mom_off, mo, &b))) { drop(); return rc; }
        if (cudaMalloc((void **)&c->d_ccout, out_bytes) != cudaSuccess || cudaMalloc((void **)&c->d_w, NROW * sizeof(float)) != cudaSuccess ||
            cudaMalloc((void **)&c->d_mom, (size_t)std::max<int64_t>(n, 1) * sizeof(double)) != cudaSuccess) {
            drop();
            return CS_ENOMEM;
        }
        c->cc_bytes = b + n * (int64_t)sizeof(double) + (int64_t)out_bytes + NROW * 4;
        c->batch_bytes += c->cc_bytes;
    }
    CK(cudaMemcpyAsync(c->d_w, c->kc.w, NROW * sizeof(float), cudaMemcpyHostToDevice, st));
    for (size_t j = 0; j < c->jobs.size(); j += 65535) {
        const int nj = (int)std::min<size_t>(65535, c->jobs.size() - j);
        dim3 grid((c->ncell_max + 3) / 4, nj);
        k_cc_moments<<<grid, 128, 0, st>>>(c->d_copy, c->nfreq, c->d_cells, c->d_momjobs + j, c->d_w, c->d_mom);
        c->launches++;
    }
    CK(cudaGetLastError());
    c->have_moments = true;
    return CS_OK;
    CS_GUARD_END
}

int cs_spectral_like_grad_cells(cs_ctx *c, double *nll, double *grad, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!nll || !c->tables_built || !c->have_moments) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    for (int e0 = 0; e0 < c->batch; e0 += 65535) {
        const int nb = std::min(65535, c->batch - e0);
        dim3 g1((c->ncell_max + 127) / 128, nb);
        k_like_cc<<<g1, 128, 0, st>>>(c->d_cfgs, c->d_cells, c->d_cfg_of + e0, c->d_mom_off + e0, c->d_tab_off + e0, c->d_tab, c->d_mom, c->kc,
                                      c->nfreq, grad ? 1 : 0, c->d_ccout + (int64_t)e0 * c->cc_out_stride, c->cc_out_stride, c->d_err);
        dim3 g2((grad ? (c->ktot_max + 127) / 128 : 0) + c->nregion, nb);   // cluster blocks, then one block per region
        k_cc_reduce<<<g2, 128, 0, st>>>(c->d_cfgs, c->d_cells, c->d_cfg_of + e0, c->d_param_off + e0, c->d_ccout + (int64_t)e0 * c->cc_out_stride,
                                        c->cc_out_stride, c->nregion, grad ? 1 : 0, nll + (int64_t)e0 * c->nregion, grad);
        c->launches += 2;
    }
    CK(cudaGetLastError());
    return CS_OK;
}

int cs_cmb_variance(cs_ctx *c, double *var, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!var || !c->tables_built) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LikeParams P = base_params(c);
    if ((rc = launch_batch<MODE_CMBVAR>(c, P, st))) return rc;
    const int n = c->batch * c->nregion;
    k_cmbvar<<<(n + 127) / 128, 128, 0, st>>>(c->d_partial, c->PS, c->d_maps, c->d_cfgs, c->d_cfg_of, c->d_npix_live,
                                             c->nregion, c->batch, var);
    c->launches++;
    CK(cudaGetLastError());
    return CS_OK;
}

void cs_opt_defaults(cs_opt *o) {
    if (!o) return;
    o->iters = 200; o->ls_max = 8;
    o->lr = 0.02; o->beta1 = 0.9; o->beta2 = 0.999; o->eps = 1e-16;
    o->ls_c1 = 1e-4; o->safe_lo = 1e-15; o->safe_hi = 1e15; o->ls_noise = 1e-7; o->topk = 0.0;
    o->method = CS_METHOD_ADATOPK; o->history = 10;
}

int cs_optimize(cs_ctx *c, double *params, const double *lower, const double *upper, const cs_opt *opt, double *nll_final,
                void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!params || !lower || !upper || !opt || opt->iters < 0 || opt->ls_max < 1 || !(opt->ls_noise >= 0) || !(opt->topk >= 0.0 && opt->topk <= 1.0))
        return CS_EINVAL;
    const bool lbfgs = opt->method == CS_METHOD_LBFGS;
    if (opt->method != CS_METHOD_ADATOPK && !lbfgs) return CS_EINVAL;
    if (lbfgs && (opt->history < 1 || opt->history > LBFGS_HIST_MAX)) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // the legacy default stream cannot be captured into a graph: fork onto an internal stream and join at the end
    cudaStream_t caller = st;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    const bool forked = (st == nullptr || st == cudaStreamLegacy);
    if (forked) {
        if (!c->comp_stream) CK(cudaStreamCreateWithFlags(&c->comp_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ev_join, cudaEventDisableTiming));
        CK(cudaEventRecord(ev_fork, caller));
        CK(cudaStreamWaitEvent(c->comp_stream, ev_fork, 0));
        st = c->comp_stream;
    }
    struct Join {   // runs on every return path
        bool on; cudaStream_t from, to; cudaEvent_t a, b;
        ~Join() {
            if (!on) return;
            cudaEventRecord(b, from);
            cudaStreamWaitEvent(to, b, 0);
            cudaEventDestroy(a); cudaEventDestroy(b);
        }
    } join{forked, st, caller, ev_fork, ev_join};
    if (!c->opt.y) {
        if ((rc = opt_alloc(c->opt, c->nparam, c->batch, c->nregion, &c->opt_bytes))) return rc == 1 ? CS_ENOMEM : CS_ECUDA;
    }
    OptShape sh{c->nparam, c->batch, c->nregion, c->ktot_max, c->d_param_off};
    OptHyper hy{opt->lr, opt->beta1, opt->beta2, opt->eps, opt->ls_c1, opt->safe_lo, opt->safe_hi, opt->ls_noise, opt->topk, opt->ls_max};
    OptWork &w = c->opt;
    if (lbfgs) {
        if (opt_alloc_lbfgs(w, c->nparam, c->batch, opt->history, &c->opt_bytes)) return CS_ENOMEM;
        lb_init(w, sh, params, lower, upper, 1e-6, st);
    } else {
        opt_init(w, sh, params, lower, upper, st);
    }
    c->launches += 1;
    // the line search compares 1/2 chi^2 of the GLS residual (cs_spectral_misfit): its value at the start
    if ((rc = cs_build_sed_tables(c, w.x, st))) return rc;
    if ((rc = cs_spectral_misfit(c, w.nll_reg_t, st))) return rc;
    opt_set_L(w, sh, st); c->launches += 1;
    // one iteration of Alg. 1; nothing in it depends on the host (the iteration counter lives on the device)
    auto iteration = [&]() -> int {
        int r;
        // value + gradient at the current point x
        if ((r = cs_build_sed_tables(c, w.x, st))) return r;
        if ((r = cs_spectral_like_grad(c, w.nll_reg, w.grad, st))) return r;
        if (lbfgs) lb_direction(w, sh, opt->history, 1e-10, st); else opt_direction(w, sh, hy, st);
        c->launches += 1;
        for (int ls = 0; ls < opt->ls_max; ++ls) {
            if (lbfgs) lb_trial_point(w, sh, st); else opt_trial_point(w, sh, st);
            c->launches += 1;
            c->skip = w.accepted;   // entries that already accepted a step sit this trial out
            r = cs_build_sed_tables(c, w.xt, st);
            if (!r) r = cs_spectral_misfit(c, w.nll_reg_t, st);
            c->skip = nullptr;
            if (r) return r;
            opt_ls_update(w, sh, hy, st); c->launches += 1;
        }
        if (lbfgs) lb_commit(w, sh, st); else opt_commit(w, sh, st);
        c->launches += 1;
        return CS_OK;
    };
    // The body is captured once into a CUDA graph and replayed: a step of a small batch is launch-bound (config 2:
    // ~30 kernels of a few microseconds each).  If the caller's stream is itself being captured, or the fused-kernel
    // timer is on, the kernels are enqueued directly.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    cudaStreamIsCapturing(st, &cap);
    bool replayed = false;
    if (opt->iters > 1 && cap == cudaStreamCaptureStatusNone && !c->prof_on) {
        if (opt->iters > 0 && (rc = iteration())) return rc;     // first iteration directly: warms up
        const int64_t l0 = c->launches;
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const int r = iteration();
            const cudaError_t ce = cudaStreamEndCapture(st, &graph);
            if (r == CS_OK && ce == cudaSuccess && graph && cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess) {
                const int64_t per_iter = c->launches - l0;
                for (int it = 1; it < opt->iters; ++it) CK(cudaGraphLaunch(exec, st));
                c->launches = l0 + per_iter * (opt->iters - 1);
                replayed = true;
            }
            if (exec) cudaGraphExecDestroy(exec);
            if (graph) cudaGraphDestroy(graph);
            if (!replayed) c->launches = l0;
        }
        if (!replayed) cudaGetLastError();
        if (!replayed)
            for (int it = 1; it < opt->iters; ++it)
                if ((rc = iteration())) return rc;
    } else {
        for (int it = 0; it < opt->iters; ++it)
            if ((rc = iteration())) return rc;
    }
    // final objective at the result
    if ((rc = cs_build_sed_tables(c, w.x, st))) return rc;
    if ((rc = cs_spectral_like_grad(c, w.nll_reg, nullptr, st))) return rc;
    opt_finish(w, sh, params, nll_final, st); c->launches += 1;
    CK(cudaGetLastError());
    return CS_OK;
}

int cs_eval_host(cs_ctx *c, int32_t ndata, const float *d_host, const float *ninv_host, const double *params_host,
                 double *nll_host, double *grad_host) {
    if (!c || c->batch <= 0 || c->maps.empty() || !d_host || !ninv_host || !params_host || !nll_host || ndata <= 0) return CS_EINVAL;
    for (int32_t e = 0; e < c->batch; ++e)
        if (c->data_of[e] >= ndata || (e > 0 && c->data_of[e] < c->data_of[e - 1])) return CS_EINVAL;
    CS_GUARD_BEGIN
    const int64_t per = (int64_t)c->nfreq * 2 * c->npix;
    const int64_t need = per * ndata * (int64_t)sizeof(float);
    if (c->stage_bytes < need) {
        cudaFree(c->d_stage);
        c->d_stage = nullptr; c->stage_bytes = 0;
        if (cudaMalloc((void **)&c->d_stage, (size_t)need) != cudaSuccess) return CS_ENOMEM;
        c->stage_bytes = need;
    }
    if (!c->d_hparams) {
        if (cudaMalloc((void **)&c->d_hparams, sizeof(double) * std::max<int64_t>(c->nparam, 1)) != cudaSuccess ||
            cudaMalloc((void **)&c->d_hgrad, sizeof(double) * std::max<int64_t>(c->nparam, 1)) != cudaSuccess ||
            cudaMalloc((void **)&c->d_hnll, sizeof(double) * c->batch * c->nregion) != cudaSuccess)
            return CS_ENOMEM;
        c->hbuf_bytes = 2 * (int64_t)sizeof(double) * c->nparam + (int64_t)sizeof(double) * c->batch * c->nregion;
    }
    if (!c->copy_stream) CK(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    if (!c->comp_stream) CK(cudaStreamCreateWithFlags(&c->comp_stream, cudaStreamNonBlocking));
    int rc = set_data_impl(c, ndata, c->d_stage, ninv_host, false);   // the staged copy becomes the context's data
    if (rc) return rc;
    cudaStream_t cp = c->copy_stream, cm = c->comp_stream;
    // parameters and tables on the compute stream while the first data chunk is in flight on the copy stream
    CK(cudaMemcpyAsync(c->d_hparams, params_host, sizeof(double) * c->nparam, cudaMemcpyHostToDevice, cm));
    if ((rc = cs_build_sed_tables(c, c->d_hparams, cm))) return rc;
    // Upload in chunks of data sets; after each chunk, on the compute stream and behind an event: gather the private
    // copies of the data sets that arrived, then run the entries whose data are resident, so that the next chunk's
    // copy overlaps their kernels.  data_of is non-decreasing, so inside every run the entries of a chunk are a
    // contiguous stretch.
    const int64_t chunk_sets = std::max<int64_t>(1, (int64_t)(128ll << 20) / (per * 4));
    const int64_t nchunk = (ndata + chunk_sets - 1) / chunk_sets;
    const int64_t nrun_all = (int64_t)c->runs.size();
    if (c->hruns_cap < nchunk * nrun_all) {
        cudaFree(c->d_hruns);
        c->d_hruns = nullptr; c->hruns_cap = 0;
        if (cudaMalloc((void **)&c->d_hruns, sizeof(Run) * (size_t)(nchunk * nrun_all)) != cudaSuccess) return CS_ENOMEM;
        c->hruns_cap = nchunk * nrun_all;
    }
    std::vector<Run> hr((size_t)(nchunk * nrun_all));
    std::vector<int32_t> cnt_sc(nchunk, 0), cnt_dir(nchunk, 0);
    std::vector<int64_t> Wsc(nchunk, 0), Wdir(nchunk, 0);
    for (int64_t ch = 0; ch < nchunk; ++ch) {
        const int64_t n0 = ch * chunk_sets, n1 = std::min<int64_t>(ndata, n0 + chunk_sets);
        Run *out = hr.data() + ch * nrun_all;
        for (int pass = 0; pass < 2; ++pass)
            for (int64_t r = 0; r < nrun_all; ++r) {
                const Run &run = c->runs[r];
                const bool sc = r < c->nrun_sc;
                if (sc != (pass == 0)) continue;
                int32_t a = run.estart, b = run.estart + run.count;
                while (a < b && c->data_of[c->elist[a]] < n0) ++a;
                int32_t e2 = a;
                while (e2 < b && c->data_of[c->elist[e2]] < n1) ++e2;
                if (e2 == a) continue;
                int64_t &W = sc ? Wsc[ch] : Wdir[ch];
                out[cnt_sc[ch] + cnt_dir[ch]] = Run{run.cfg, a, e2 - a, run.ntile, W, run.hdr, run.hdrptr, run.tstride};
                W += (int64_t)run.ntile * (e2 - a);
                (sc ? cnt_sc[ch] : cnt_dir[ch])++;
            }
    }
    CK(cudaMemcpyAsync(c->d_hruns, hr.data(), sizeof(Run) * hr.size(), cudaMemcpyHostToDevice, cm));
    LikeParams P = base_params(c);
    std::vector<cudaEvent_t> evs;
    rc = CS_OK;
    size_t j0 = 0;
    for (int64_t ch = 0; ch < nchunk && rc == CS_OK; ++ch) {
        const int64_t n0 = ch * chunk_sets, n1 = std::min<int64_t>(ndata, n0 + chunk_sets);
        cudaEvent_t ev;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { rc = CS_ECUDA; break; }
        evs.push_back(ev);
        if (cudaMemcpyAsync(c->d_stage + n0 * per, d_host + n0 * per, (size_t)((n1 - n0) * per) * sizeof(float),
                            cudaMemcpyHostToDevice, cp) != cudaSuccess ||
            cudaEventRecord(ev, cp) != cudaSuccess || cudaStreamWaitEvent(cm, ev, 0) != cudaSuccess) { rc = CS_ECUDA; break; }
        size_t j1 = j0;
        while (j1 < c->jobs.size() && c->jobs[j1].data < n1) ++j1;
        if (j1 > j0) rc = relayout(c, c->d_stage, (int64_t)j0, (int64_t)j1, cm);
        j0 = j1;
        if (rc == CS_OK && cnt_sc[ch] + cnt_dir[ch] > 0) {
            const Run *dr = c->d_hruns + ch * nrun_all;
            rc = grad_host ? launch_like<MODE_GRAD>(c, P, dr, cnt_sc[ch], Wsc[ch], cnt_dir[ch], Wdir[ch], cm)
                           : launch_like<MODE_VALUE>(c, P, dr, cnt_sc[ch], Wsc[ch], cnt_dir[ch], Wdir[ch], cm);
        }
    }
    if (rc == CS_OK) rc = merge_launch(c, c->d_hnll, grad_host ? c->d_hgrad : nullptr, cm);
    if (rc == CS_OK && cudaMemcpyAsync(nll_host, c->d_hnll, sizeof(double) * c->batch * c->nregion, cudaMemcpyDeviceToHost, cm) != cudaSuccess) rc = CS_ECUDA;
    if (rc == CS_OK && grad_host && cudaMemcpyAsync(grad_host, c->d_hgrad, sizeof(double) * c->nparam, cudaMemcpyDeviceToHost, cm) != cudaSuccess) rc = CS_ECUDA;
    if (cudaStreamSynchronize(cp) != cudaSuccess || cudaStreamSynchronize(cm) != cudaSuccess) rc = rc ? rc : CS_ECUDA;
    for (cudaEvent_t ev : evs) cudaEventDestroy(ev);
    return rc;
    CS_GUARD_END
}

int cs_spherical_kmeans(int64_t npix, const double *vecs, const uint8_t *region, int32_t nprob, const int32_t *K,
                        const int32_t *prob_region, double *cent, int32_t iters, int32_t *labels, void *stream) {
    if (npix <= 0 || !vecs || nprob <= 0 || !K || !cent || iters < 0 || !labels) return CS_EINVAL;
    CS_GUARD_BEGIN
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<KmProb> pr(nprob);
    int64_t off = 0;
    for (int32_t j = 0; j < nprob; ++j) {
        if (K[j] < 1) return CS_EINVAL;
        const int32_t reg = prob_region ? prob_region[j] : -1;
        if (reg >= 0 && !region) return CS_EINVAL;
        pr[j] = KmProb{K[j], reg, off};
        off += K[j];
    }
    KmProb *d_pr = nullptr;
    if (cudaMallocAsync((void **)&d_pr, sizeof(KmProb) * nprob, st) != cudaSuccess) return CS_ENOMEM;
    // pageable host memory: the copy has left the host buffer when cudaMemcpyAsync returns
    if (cudaMemcpyAsync(d_pr, pr.data(), sizeof(KmProb) * nprob, cudaMemcpyHostToDevice, st) != cudaSuccess) { cudaFreeAsync(d_pr, st); return CS_ECUDA; }
    // problems are independent: more than 65535 of them (the limit of grid.y) go in slices, one after the other
    for (int32_t j0 = 0; j0 < nprob; j0 += 65535) {
        const int32_t nj = std::min<int32_t>(65535, nprob - j0);
        int32_t kmax_j = 0;
        for (int32_t j = j0; j < j0 + nj; ++j) kmax_j = std::max(kmax_j, K[j]);
        const dim3 ga((unsigned)((npix + 255) / 256), nj), gu((kmax_j + 7) / 8, nj);
        int32_t *lab_j = labels + (int64_t)j0 * npix;
        k_km_assign<<<ga, 256, 0, st>>>(vecs, npix, region, d_pr + j0, cent, lab_j);
        for (int32_t it = 0; it < iters; ++it) {
            k_km_update<<<gu, 256, 0, st>>>(vecs, npix, d_pr + j0, lab_j, cent);
            k_km_assign<<<ga, 256, 0, st>>>(vecs, npix, region, d_pr + j0, cent, lab_j);
        }
    }
    const cudaError_t ce = cudaGetLastError();
    cudaFreeAsync(d_pr, st);
    return ce == cudaSuccess ? CS_OK : CS_ECUDA;
    CS_GUARD_END
}

int cs_check(cs_ctx *c, void *stream) {
    if (!c) return CS_EINVAL;
    CK(cudaStreamSynchronize((cudaStream_t)stream));
    int32_t e = 0;
    CK(cudaMemcpy(&e, c->d_err, sizeof(e), cudaMemcpyDeviceToHost));
    CK(cudaMemset(c->d_err, 0, sizeof(e)));
    if (e & ERR_DOMAIN) return CS_EDOMAIN;
    if (e & ERR_SINGULAR) return CS_ESINGULAR;
    return CS_OK;
}

int cs_profile(cs_ctx *c, int enable) {
    if (!c) return CS_EINVAL;
    if (enable && c->prof_ev.empty()) {
        c->prof_ev.resize(2 * cs_ctx::PROF_RING);
        for (auto &e : c->prof_ev) CK(cudaEventCreate(&e));
    }
    c->prof_on = enable != 0;
    c->prof_n = 0;
    return CS_OK;
}

int cs_profile_read(cs_ctx *c, double *total_ms, int64_t *count) {
    if (!c || !total_ms || !count) return CS_EINVAL;
    CK(cudaDeviceSynchronize());
    const int64_t n = std::min<int64_t>(c->prof_n, cs_ctx::PROF_RING);
    double tot = 0;
    for (int64_t i = 0; i < n; ++i) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
        tot += ms;
    }
    *total_ms = tot; *count = n;
    return CS_OK;
}

int64_t cs_workspace_bytes(cs_ctx *c) {
    if (!c) return 0;
    return c->cluster_bytes + c->batch_bytes + c->opt_bytes + c->stage_bytes + c->hbuf_bytes;
}

int64_t cs_kernel_launches(cs_ctx *c) { return c ? c->launches : 0; }

}  // extern "C"

// ---- cs_spherical_kmeans_static: the K-means entry point that allocates nothing (include/cs.h) -------------------------
// The problem descriptors that cs_spherical_kmeans puts in a cudaMallocAsync'ed table live here instead, in the library
// image: 1024 x 16 B = 16 KiB on every GPU that loads libcs.so, until the process exits.  On the host the name
// g_km_static_probs is only a handle for the runtime's symbol calls, not an address a kernel can use; the launches
// below get the device address that km_static_table() looks up.
static __device__ __align__(256) KmProb g_km_static_probs[CS_KMEANS_STATIC_MAX_PROB];

namespace {
constexpr int KM_STATIC_MAX_DEV = 64;
std::mutex g_km_static_mu;
KmProb *g_km_static_addr[KM_STATIC_MAX_DEV] = {};

// Device address of g_km_static_probs on the current device; asked of the runtime once per device, with that device
// current, and kept.  Every device has its own copy of the array at its own address.
int km_static_table(KmProb **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= KM_STATIC_MAX_DEV) return CS_ECUDA;
    std::lock_guard<std::mutex> lock(g_km_static_mu);
    if (!g_km_static_addr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_km_static_probs) != cudaSuccess || !p) return CS_ECUDA;
        g_km_static_addr[dev] = (KmProb *)p;
    }
    *out = g_km_static_addr[dev];
    return CS_OK;
}
}  // namespace

extern "C" int cs_spherical_kmeans_static(int64_t npix, const double *vecs, const uint8_t *region, int32_t nprob, const int32_t *K,
                                          const int32_t *prob_region, double *cent, int32_t iters, int32_t *labels, void *stream) {
    if (npix <= 0 || !vecs || nprob <= 0 || !K || !cent || iters < 0 || !labels) return CS_EINVAL;
    if (nprob > CS_KMEANS_STATIC_MAX_PROB) return CS_ELIMIT;
    cudaStream_t st = (cudaStream_t)stream;
    KmProb pr[CS_KMEANS_STATIC_MAX_PROB];   // host staging on the stack: no heap either
    int64_t off = 0;
    int32_t kmax = 0;
    for (int32_t j = 0; j < nprob; ++j) {
        if (K[j] < 1) return CS_EINVAL;
        const int32_t reg = prob_region ? prob_region[j] : -1;
        if (reg >= 0 && !region) return CS_EINVAL;
        pr[j] = KmProb{K[j], reg, off};
        off += K[j];
        kmax = std::max(kmax, K[j]);
    }
    KmProb *d_pr = nullptr;
    const int rc = km_static_table(&d_pr);
    if (rc != CS_OK) return rc;
    // Overwrites the descriptors this call reads, in stream order: earlier calls on `st` have finished with the table
    // by then.  Pageable source: the bytes have left `pr` when cudaMemcpyAsync returns.
    if (cudaMemcpyAsync(d_pr, pr, sizeof(KmProb) * nprob, cudaMemcpyHostToDevice, st) != cudaSuccess) return CS_ECUDA;
    const dim3 ga((unsigned)((npix + 255) / 256), nprob), gu((kmax + 7) / 8, nprob);
    k_km_assign<<<ga, 256, 0, st>>>(vecs, npix, region, d_pr, cent, labels);
    for (int32_t it = 0; it < iters; ++it) {
        k_km_update<<<gu, 256, 0, st>>>(vecs, npix, d_pr, labels, cent);
        k_km_assign<<<ga, 256, 0, st>>>(vecs, npix, region, d_pr, cent, labels);
    }
    return cudaGetLastError() == cudaSuccess ? CS_OK : CS_ECUDA;
}
