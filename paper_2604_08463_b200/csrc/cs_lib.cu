// cs_lib.cu -- C ABI of libcs (include/cs.h): context, reduction plan, launches.  No CPU compute path exists:
// every arithmetic step of the hot path runs in the kernels of cs_kernels.cuh; the host code below only
// validates, builds index structures once per clustering and launches.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cs.h"
#include "cs_kernels.cuh"
#include "cs_like_cell.cuh"
#include "cs_optim.cuh"

using namespace cs;

#define CK(call)                                   \
    do {                                           \
        cudaError_t err__ = (call);                \
        if (err__ != cudaSuccess) return CS_ECUDA; \
    } while (0)

namespace {

struct MapHost {
    int32_t K = 0, nseg = 0;
    int32_t *idx = nullptr;
    uint8_t *rank = nullptr;
    int32_t *segptr = nullptr;
    uint16_t *segdesc = nullptr;
    int32_t *segslot = nullptr;
    int32_t *ksegptr = nullptr;
    int32_t *chunkptr = nullptr;
    uint16_t *segcfirst = nullptr;
    std::vector<int32_t> h_chunkptr, h_segptr;   // host copies: per-tile counts decide a configuration's kernel
};

// Device arrays of one configuration's cell plan (empty when it runs on the direct kernel).
struct CellHost {
    uint8_t *cellid = nullptr;
    int32_t *cellptr = nullptr;
    int32_t *cellrows = nullptr;
    int32_t *rowptr = nullptr;
    int32_t *rowlist = nullptr;
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

}  // namespace

struct cs_ctx {
    // model
    int32_t nfreq = 0, units = 0;
    int64_t npix = 0;
    int32_t ntile = 0;
    double freqs[NROW] = {0};
    double nu0d = 0, nu0s = 0, tcmb = 0;
    TConst tc;
    KConst kc;
    bool have_ninv = false;
    // clusters
    int32_t nmap = 0, ncfg = 0, nregion = 1;
    std::vector<MapHost> maps;          // nmap + 1 (last = region pseudo-map)
    std::vector<CfgDev> cfgs;
    std::vector<CellHost> cellplans;    // ncfg
    std::vector<int32_t> npix_live;     // [ncfg*nregion]
    MapDev *d_maps = nullptr;
    CfgDev *d_cfgs = nullptr;
    int32_t *d_npix_live = nullptr;
    int64_t cluster_bytes = 0;
    // data
    const float *d = nullptr;
    int32_t ndata = 0;
    CUtensorMap tmap;                   // d as [ndata*2*nfreq, npix], box [2*nfreq, 32]   (direct kernel: one box per warp)
    CUtensorMap tmap_cta;               // same tensor, box [2*nfreq, TP]                  (cell kernel: one box per CTA)
    bool have_tmap = false;
    // batch
    int32_t batch = 0, ngroup = 0, ngroup_cell = 0, ktot_max = 0;   // groups [0, ngroup_cell) run on the cell kernel
    int64_t nparam = 0, nrows = 0, PS = 0;
    std::vector<int32_t> cfg_of, data_of;
    std::vector<int64_t> param_off;
    int32_t *d_cfg_of = nullptr, *d_data_of = nullptr, *d_elist = nullptr, *d_sel_elist = nullptr;
    int64_t *d_param_off = nullptr, *d_tab_off = nullptr;
    Group *d_groups = nullptr, *d_sel_groups = nullptr;
    float *d_tab = nullptr;
    double *d_partial = nullptr;
    int64_t batch_bytes = 0;
    // optimizer workspace
    OptWork opt;
    int64_t opt_bytes = 0;
    // host-eval staging
    float *d_stage = nullptr;
    int64_t stage_bytes = 0;
    double *d_hparams = nullptr, *d_hnll = nullptr, *d_hgrad = nullptr;
    int64_t hbuf_bytes = 0;
    cudaStream_t copy_stream = nullptr, comp_stream = nullptr;
    // optional timing of the fused kernel (cs_profile): ring of event pairs recorded around every k_like launch
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
    int32_t cell_min_group = CELL_MIN_GROUP;   // CS_CELL_MIN_GROUP overrides (tests run the cell kernel on 1-entry groups)
    bool force_direct = false;          // CS_FORCE_DIRECT=1 in the environment at cs_create: never use the cell kernel (tests)
};

namespace {

void free_clusters(cs_ctx *c) {
    for (auto &m : c->maps) {
        cudaFree(m.idx); cudaFree(m.rank); cudaFree(m.segptr); cudaFree(m.segdesc); cudaFree(m.segslot); cudaFree(m.ksegptr);
        cudaFree(m.chunkptr); cudaFree(m.segcfirst);
    }
    c->maps.clear();
    for (auto &p : c->cellplans) { cudaFree(p.cellid); cudaFree(p.cellptr); cudaFree(p.cellrows); cudaFree(p.rowptr); cudaFree(p.rowlist); }
    c->cellplans.clear();
    cudaFree(c->d_maps); cudaFree(c->d_cfgs); cudaFree(c->d_npix_live);
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
    cudaFree(c->d_cfg_of); cudaFree(c->d_data_of); cudaFree(c->d_elist); cudaFree(c->d_sel_elist);
    cudaFree(c->d_param_off); cudaFree(c->d_tab_off); cudaFree(c->d_groups); cudaFree(c->d_sel_groups);
    cudaFree(c->d_tab); cudaFree(c->d_partial);
    c->d_cfg_of = c->d_data_of = c->d_elist = c->d_sel_elist = nullptr;
    c->d_param_off = c->d_tab_off = nullptr;
    c->d_groups = c->d_sel_groups = nullptr;
    c->d_tab = nullptr; c->d_partial = nullptr;
    c->batch = 0; c->ngroup = 0; c->batch_bytes = 0;
    c->tables_built = false;
    cudaFree(c->d_hparams); cudaFree(c->d_hnll); cudaFree(c->d_hgrad);
    c->d_hparams = c->d_hnll = c->d_hgrad = nullptr;
    c->hbuf_bytes = 0;
    free_opt(c);
}

// K_RJ -> K_CMB factor u(nu) = (e^x - 1)^2 / (x^2 e^x), x = h nu / (k_B T_cmb)   (R2)
double krj2kcmb(double nu_ghz, double tcmb, double hk) {
    const double x = hk * nu_ghz / tcmb;
    const double em1 = std::expm1(x);
    return em1 * em1 / (x * x * std::exp(x));
}

// Reduction plan of one cluster map: per tile the rank of every pixel in the (cluster, pixel) order, that order cut
// into segments of <= SEG_MAX pixels of one cluster, plus the CSR cluster -> segments.
int build_map_plan(const int32_t *idx, int32_t K, int64_t npix, int32_t ntile, MapHost *out, int64_t *bytes) {
    std::vector<uint8_t> rank((size_t)ntile * TP, 0);
    std::vector<int32_t> segptr(ntile + 1, 0);
    std::vector<uint16_t> segdesc;
    std::vector<int32_t> segcluster;
    segdesc.reserve((size_t)ntile * 16);
    segcluster.reserve((size_t)ntile * 16);
    std::vector<std::pair<int32_t, int32_t>> tmp;
    std::vector<std::pair<uint16_t, int32_t>> tseg;   // (descriptor, cluster)
    std::vector<int32_t> chunkptr(ntile + 1, 0);
    std::vector<uint16_t> segcfirst;
    int32_t nchunk = 0;
    tmp.reserve(TP);
    for (int32_t t = 0; t < ntile; ++t) {
        tmp.clear();
        const int64_t p0 = (int64_t)t * TP;
        const int nv = (int)std::min<int64_t>(TP, npix - p0);
        for (int j = 0; j < nv; ++j)
            if (idx[p0 + j] >= 0) tmp.emplace_back(idx[p0 + j], j);
        std::sort(tmp.begin(), tmp.end());
        segptr[t] = (int32_t)segdesc.size();
        // segments of this tile, longest first: the lanes of a warp of the reduce phase then walk runs of similar length
        tseg.clear();
        size_t i = 0;
        while (i < tmp.size()) {
            size_t j = i;
            while (j < tmp.size() && tmp[j].first == tmp[i].first && j - i < (size_t)SEG_MAX) ++j;
            tseg.push_back({(uint16_t)(i | ((j - i - 1) << 8)), tmp[i].first});
            i = j;
        }
        std::stable_sort(tseg.begin(), tseg.end(), [](const std::pair<uint16_t, int32_t> &a, const std::pair<uint16_t, int32_t> &b) {
            return (a.first >> 8) > (b.first >> 8);
        });
        chunkptr[t] = nchunk;
        int32_t local = 0;
        for (auto &sg : tseg) {
            segdesc.push_back(sg.first); segcluster.push_back(sg.second);
            segcfirst.push_back((uint16_t)local);
            local += ((sg.first >> 8) + 1 + CHUNK_LEN - 1) / CHUNK_LEN;
        }
        nchunk += local;
        for (size_t q = 0; q < tmp.size(); ++q) rank[p0 + tmp[q].second] = (uint8_t)q;
    }
    segptr[ntile] = (int32_t)segdesc.size();
    chunkptr[ntile] = nchunk;
    const int32_t nseg = (int32_t)segdesc.size();
    // cluster-major slots: the segments of cluster k occupy [ksegptr[k], ksegptr[k+1]) in ascending (tile, chunk) order
    std::vector<int32_t> ksegptr(K + 1, 0), segslot(nseg);
    for (int32_t s = 0; s < nseg; ++s) ksegptr[segcluster[s] + 1]++;
    for (int32_t k = 0; k < K; ++k) ksegptr[k + 1] += ksegptr[k];
    std::vector<int32_t> fill(ksegptr.begin(), ksegptr.end() - 1);
    for (int32_t s = 0; s < nseg; ++s) segslot[s] = fill[segcluster[s]]++;
    std::vector<int32_t> idxv(idx, idx + npix);
    out->K = K; out->nseg = nseg;
    int rc;
    if ((rc = dev_upload(&out->idx, idxv, bytes))) return rc;
    if ((rc = dev_upload(&out->rank, rank, bytes))) return rc;
    if ((rc = dev_upload(&out->segptr, segptr, bytes))) return rc;
    if ((rc = dev_upload(&out->segdesc, segdesc, bytes))) return rc;
    if ((rc = dev_upload(&out->segslot, segslot, bytes))) return rc;
    if ((rc = dev_upload(&out->ksegptr, ksegptr, bytes))) return rc;
    if ((rc = dev_upload(&out->chunkptr, chunkptr, bytes))) return rc;
    if ((rc = dev_upload(&out->segcfirst, segcfirst, bytes))) return rc;
    out->h_chunkptr = chunkptr; out->h_segptr = segptr;
    return CS_OK;
}

// Cell plan of one configuration: per tile the distinct (k0,k1,k2) triples in order of first appearance, as table-row
// indices of an entry's table block.  Returns 1 (and uploads nothing) when some tile holds more than CELL_CAP cells:
// that configuration then runs on the direct kernel.
int build_cell_plan(const int32_t *i0, const int32_t *i1, const int32_t *i2, const int32_t K[3], int64_t npix, int32_t ntile,
                    CellHost *out, int32_t *ncell_max, int64_t *bytes) {
    std::vector<uint8_t> cellid((size_t)ntile * TP, 0xFF);
    std::vector<int32_t> cellptr(ntile + 1, 0);
    std::vector<int32_t> rows, rowlist, rowptr(ntile + 1, 0);
    rows.reserve((size_t)ntile * 64 * 4);
    int32_t mx = 0;
    for (int32_t t = 0; t < ntile; ++t) {
        const int64_t p0 = (int64_t)t * TP;
        const int nv = (int)std::min<int64_t>(TP, npix - p0);
        const size_t base = rows.size() / 4;
        cellptr[t] = (int32_t)base;
        int n = 0, last = -1;
        for (int j = 0; j < nv; ++j) {
            const int32_t a = i0[p0 + j], b = i1[p0 + j], d = i2[p0 + j];
            if (a < 0 || b < 0 || d < 0) continue;
            const int32_t r0 = a, r1 = K[0] + b, r3 = K[0] + 2 * K[1] + d;
            int id = -1;
            if (last >= 0 && rows[4 * (base + last)] == r0 && rows[4 * (base + last) + 1] == r1 && rows[4 * (base + last) + 3] == r3) {
                id = last;   // consecutive pixels mostly share their cell
            } else {
                for (int q = n - 1; q >= 0; --q)
                    if (rows[4 * (base + q)] == r0 && rows[4 * (base + q) + 1] == r1 && rows[4 * (base + q) + 3] == r3) { id = q; break; }
            }
            if (id < 0) {
                if (n == CELL_CAP) return 1;
                id = n++;
                rows.push_back(r0); rows.push_back(r1); rows.push_back(K[0] + K[1] + b); rows.push_back(r3);
            }
            cellid[p0 + j] = (uint8_t)id;
            last = id;
        }
        mx = std::max(mx, n);
        // the tile's distinct table rows; cells keep slots into this list (the loader stages the list per entry)
        rowptr[t] = (int32_t)rowlist.size();
        const size_t r0 = rowlist.size();
        for (size_t q = 4 * base; q < rows.size(); ++q) {
            size_t f = r0;
            while (f < rowlist.size() && rowlist[f] != rows[q]) ++f;
            if (f == rowlist.size()) {
                if (rowlist.size() - r0 == (size_t)ROW_CAP) return 1;
                rowlist.push_back(rows[q]);
            }
            rows[q] = (int32_t)(f - r0);
        }
    }
    rowptr[ntile] = (int32_t)rowlist.size();
    cellptr[ntile] = (int32_t)(rows.size() / 4);
    *ncell_max = mx;
    int rc;
    if ((rc = dev_upload(&out->cellid, cellid, bytes))) return rc;
    if ((rc = dev_upload(&out->cellptr, cellptr, bytes))) return rc;
    if ((rc = dev_upload(&out->cellrows, rows, bytes))) return rc;
    if ((rc = dev_upload(&out->rowptr, rowptr, bytes))) return rc;
    if ((rc = dev_upload(&out->rowlist, rowlist, bytes))) return rc;
    return CS_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// TMA descriptor of d viewed as a 2-D fp32 tensor [ndata*2*nfreq rows, npix]; one box = all rows of one data set for
// 32 consecutive pixels.  Only possible when rows are 16-byte aligned; otherwise the kernels use plain loads.
int make_tmap(cs_ctx *c) {
    c->have_tmap = false;
    std::memset(&c->tmap, 0, sizeof(c->tmap));
    std::memset(&c->tmap_cta, 0, sizeof(c->tmap_cta));
    if ((c->npix % 4) != 0 || (((uintptr_t)c->d) % 16) != 0) return CS_OK;
    static EncodeTiledFn enc = nullptr;
    if (!enc) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return CS_ECUDA;
        enc = (EncodeTiledFn)fn;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)c->npix, (cuuint64_t)c->ndata * 2 * c->nfreq};
    const cuuint64_t strides[1] = {(cuuint64_t)c->npix * 4};
    const cuuint32_t box[2] = {32, (cuuint32_t)(2 * c->nfreq)}, es[2] = {1, 1};
    if (enc(&c->tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)c->d, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return CS_ECUDA;
    const cuuint32_t box_cta[2] = {(cuuint32_t)TP, (cuuint32_t)(2 * c->nfreq)};
    if (enc(&c->tmap_cta, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)c->d, dims, strides, box_cta, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return CS_ECUDA;
    c->have_tmap = true;
    return CS_OK;
}

// Launches the fused kernel over the groups [g0, g1) of P.groups; groups below `ncell` (cell path) run on
// k_like_cell, the rest on the direct kernel k_like.  grid.y is limited to 65535: launch in slabs of groups.
template <int NF, int MODE>
int launch_like_t(cs_ctx *c, const LikeParams &P, int g0, int g1, int ncell, cudaStream_t st) {
    static bool configured = false;
    constexpr size_t smem = like_smem_bytes<NF>(), smem_cell = cell_smem_bytes<NF>();
    if (!configured) {
        CK(cudaFuncSetAttribute(k_like<NF, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CK(cudaFuncSetAttribute(k_like_cell<NF, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cell));
        configured = true;
    }
    const bool prof = c->prof_on && MODE == MODE_GRAD;
    for (int pass = 0; pass < 2; ++pass) {
        const int a = pass == 0 ? g0 : std::max(g0, ncell), b = pass == 0 ? std::min(g1, ncell) : g1;
        for (int g = a; g < b; g += 65535) {
            LikeParams Q = P;
            Q.groups = P.groups + g;
            dim3 grid(c->ntile, std::min(65535, b - g));
            if (prof) cudaEventRecord(c->prof_ev[2 * (c->prof_n % cs_ctx::PROF_RING)], st);
            if (pass == 0) k_like_cell<NF, MODE><<<grid, CELL_THREADS, smem_cell, st>>>(c->tmap_cta, Q);
            else k_like<NF, MODE><<<grid, TP, smem, st>>>(c->tmap, Q);
            if (prof) { cudaEventRecord(c->prof_ev[2 * (c->prof_n % cs_ctx::PROF_RING) + 1], st); c->prof_n++; }
            c->launches++;
        }
    }
    CK(cudaGetLastError());
    return CS_OK;
}

template <int MODE>
int launch_like(cs_ctx *c, const LikeParams &P, int g0, int g1, int ncell, cudaStream_t st) {
    if (c->nfreq == 15) return launch_like_t<15, MODE>(c, P, g0, g1, ncell, st);
    return launch_like_t<16, MODE>(c, P, g0, g1, ncell, st);
}

LikeParams base_params(cs_ctx *c) {
    LikeParams P;
    P.d = c->d;
    P.npix = c->npix;
    P.nfreq = c->nfreq;
    P.use_bulk = c->have_tmap ? 1 : 0;
    P.evict_first = ((int64_t)c->ndata * c->nfreq * 2 * c->npix * 4 > (int64_t)96 << 20) ? 1 : 0;
    P.maps = c->d_maps;
    P.cfgs = c->d_cfgs;
    P.groups = c->d_groups;
    P.elist = c->d_elist;
    P.data_of = c->d_data_of;
    P.skip = c->skip;
    P.tab_off = c->d_tab_off;
    P.tab = c->d_tab;
    P.partial = c->d_partial;
    P.PS = c->PS;
    P.maps_out = nullptr;
    P.err = c->d_err;
    P.kc = c->kc;
    return P;
}

int ready(cs_ctx *c) {
    if (!c || c->maps.empty() || !c->d || !c->have_ninv || c->batch <= 0) return CS_EINVAL;
    return CS_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------
extern "C" {

int cs_version(void) { return 1; }

const char *cs_strerror(int code) {
    switch (code) {
        case CS_OK: return "ok";
        case CS_EINVAL: return "invalid argument or call order";
        case CS_EINDEX: return "cluster or region index out of range";
        case CS_EDOMAIN: return "T_d <= 0 or non-finite spectral parameter";
        case CS_ESINGULAR: return "singular A^T N^-1 A";
        case CS_ECUDA: return "CUDA runtime error";
        case CS_ENOMEM: return "out of device memory";
        default: return "unknown error";
    }
}

int cs_create(cs_ctx **out, const cs_model *m) {
    if (!out) return CS_EINVAL;
    *out = nullptr;
    if (!m || !m->freqs_ghz || m->nfreq < 3 || m->nfreq > CS_MAX_NFREQ || m->npix <= 0 || m->npix > (int64_t)TP * 0x7fffff00)
        return CS_EINVAL;
    if (!(m->nu0_dust_ghz > 0) || !(m->nu0_sync_ghz > 0) || !(m->t_cmb_k > 0)) return CS_EINVAL;
    if (m->units != CS_UNITS_KCMB && m->units != CS_UNITS_LITERAL) return CS_EINVAL;
    for (int f = 0; f < m->nfreq; ++f)
        if (!(m->freqs_ghz[f] > 0) || !std::isfinite(m->freqs_ghz[f])) return CS_EINVAL;
    cs_ctx *c = new (std::nothrow) cs_ctx();
    if (!c) return CS_ENOMEM;
    c->nfreq = m->nfreq; c->units = m->units; c->npix = m->npix;
    c->ntile = (int32_t)((m->npix + TP - 1) / TP);
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
    if (cudaMalloc((void **)&c->d_err, sizeof(int32_t)) != cudaSuccess || cudaMemset(c->d_err, 0, sizeof(int32_t)) != cudaSuccess ||
        cudaMalloc((void **)&c->d_tc, sizeof(TConst)) != cudaSuccess ||
        cudaMemcpy(c->d_tc, &c->tc, sizeof(TConst), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaFree(c->d_err); cudaFree(c->d_tc);
        delete c;
        return CS_ECUDA;
    }
    const char *fd = std::getenv("CS_FORCE_DIRECT");
    c->force_direct = fd && fd[0] == '1';
    const char *mg = std::getenv("CS_CELL_MIN_GROUP");
    if (mg && std::atoi(mg) >= 1) c->cell_min_group = std::atoi(mg);
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
    delete c;
    return CS_OK;
}

int cs_set_clusters(cs_ctx *c, int32_t nmap, const int32_t *maps, const int32_t *Kmap, int32_t ncfg,
                    const int32_t *cfg_maps, const uint8_t *region_idx, int32_t nregion) {
    if (!c || nmap <= 0 || !maps || !Kmap || ncfg <= 0 || !cfg_maps || nregion < 1 || nregion > 255) return CS_EINVAL;
    if (nregion > 1 && !region_idx) return CS_EINVAL;
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
    c->maps.resize(nmap + 1);
    int rc;
    for (int32_t m = 0; m < nmap; ++m)
        if ((rc = build_map_plan(h.data() + (size_t)m * npix, Kmap[m], npix, c->ntile, &c->maps[m], &c->cluster_bytes))) {
            free_clusters(c);
            return rc;
        }
    if ((rc = build_map_plan(reg.data(), nregion, npix, c->ntile, &c->maps[nmap], &c->cluster_bytes))) {
        free_clusters(c);
        return rc;
    }
    c->nmap = nmap; c->ncfg = ncfg; c->nregion = nregion;
    std::vector<MapDev> md(nmap + 1);
    for (int32_t m = 0; m <= nmap; ++m) {
        const MapHost &s = c->maps[m];
        md[m] = MapDev{s.idx, s.rank, s.segptr, s.segdesc, s.segslot, s.ksegptr, s.chunkptr, s.segcfirst, s.K, s.nseg};
    }
    c->cfgs.resize(ncfg);
    c->cellplans.resize(ncfg);
    c->npix_live.assign((size_t)ncfg * nregion, 0);
    for (int32_t i = 0; i < ncfg; ++i) {
        CfgDev &cf = c->cfgs[i];
        int32_t off = 0;
        for (int t = 0; t < 4; ++t) {
            cf.map[t] = t < 3 ? cfg_maps[i * 3 + t] : nmap;
            cf.segbase[t] = off;
            off += c->maps[cf.map[t]].nseg;
            if (t < 3) cf.K[t] = Kmap[cf.map[t]];
        }
        cf.ktot = cf.K[0] + cf.K[1] + cf.K[2];
        const int32_t *a = h.data() + (size_t)cf.map[0] * npix, *b = h.data() + (size_t)cf.map[1] * npix,
                      *d = h.data() + (size_t)cf.map[2] * npix;
        for (int64_t p = 0; p < npix; ++p)
            if (a[p] >= 0 && b[p] >= 0 && d[p] >= 0) c->npix_live[(size_t)i * nregion + reg[p]]++;
        // cell plan; a configuration with a tile of more than CELL_CAP distinct triples stays on the direct kernel
        cf.cellid = nullptr; cf.cellptr = nullptr; cf.cellrows = nullptr; cf.rowptr = nullptr; cf.rowlist = nullptr;
        cf.ncell_max = 0; cf.pad = 0;
        if (!c->force_direct) {
            int32_t mx = 0;
            rc = build_cell_plan(a, b, d, cf.K, npix, c->ntile, &c->cellplans[i], &mx, &c->cluster_bytes);
            if (rc < 0) { free_clusters(c); return rc; }
            if (rc == 0) {   // the reducer warps' plan must fit too
                for (int32_t t = 0; t < c->ntile && rc == 0; ++t) {
                    int32_t nc = 0, ns = 0;
                    for (int q = 0; q < 4; ++q) {
                        const MapHost &mh = c->maps[cf.map[q]];
                        nc += mh.h_chunkptr[t + 1] - mh.h_chunkptr[t];
                        ns += mh.h_segptr[t + 1] - mh.h_segptr[t];
                    }
                    // CMBVAR reduces all four terms over the region map
                    const MapHost &mr = c->maps[cf.map[3]];
                    nc = std::max(nc, 4 * (mr.h_chunkptr[t + 1] - mr.h_chunkptr[t]));
                    if (nc > CHUNK_CAP || ns > CHUNK_CAP) rc = 1;
                }
                if (rc == 1) {
                    cudaFree(c->cellplans[i].cellid); cudaFree(c->cellplans[i].cellptr); cudaFree(c->cellplans[i].cellrows);
                    cudaFree(c->cellplans[i].rowptr); cudaFree(c->cellplans[i].rowlist);
                    c->cellplans[i] = CellHost();
                }
            }
            if (rc == 0) {
                cf.cellid = c->cellplans[i].cellid; cf.cellptr = c->cellplans[i].cellptr; cf.cellrows = c->cellplans[i].cellrows;
                cf.rowptr = c->cellplans[i].rowptr; cf.rowlist = c->cellplans[i].rowlist;
                cf.ncell_max = std::max(mx, 1);
            }
        }
    }
    if ((rc = dev_upload(&c->d_maps, md, &c->cluster_bytes)) || (rc = dev_upload(&c->d_cfgs, c->cfgs, &c->cluster_bytes)) ||
        (rc = dev_upload(&c->d_npix_live, c->npix_live, &c->cluster_bytes))) {
        free_clusters(c);
        return rc;
    }
    return CS_OK;
}

int cs_set_data(cs_ctx *c, int32_t ndata, const float *d, const float *ninv) {
    if (!c || ndata <= 0 || !d || !ninv) return CS_EINVAL;
    float w[NROW] = {0};
    CK(cudaMemcpy(w, ninv, sizeof(float) * c->nfreq, cudaMemcpyDefault));
    double m00 = 0;
    for (int f = 0; f < c->nfreq; ++f) {
        if (!(w[f] > 0.f) || !std::isfinite(w[f])) return CS_EINVAL;
        m00 += (double)w[f];
    }
    std::memset(&c->kc, 0, sizeof(c->kc));
    float m00f = 0.f;
    for (int f = 0; f < c->nfreq; ++f) {
        c->kc.w[f] = w[f];
        c->kc.lnd[f] = (float)c->tc.lnd[f];
        c->kc.lnsw[f] = (float)(c->tc.lns[f] * (double)w[f]);
        c->kc.lns[f] = (float)c->tc.lns[f];
        c->kc.invw[f] = 1.0f / w[f];
        m00f += w[f];
    }
    (void)m00f;
    c->kc.m00 = (float)m00;
    c->kc.inv_m00 = (float)(1.0 / m00);
    c->d = d;
    c->ndata = ndata;
    c->have_ninv = true;
    int rc = make_tmap(c);
    if (rc) return rc;
    for (int e = 0; e < c->batch; ++e)
        if (c->data_of[e] >= ndata) return CS_EINVAL;
    return CS_OK;
}

int cs_set_batch(cs_ctx *c, int32_t batch, const int32_t *cfg_of, const int32_t *data_of) {
    if (!c || c->maps.empty() || batch <= 0 || !cfg_of || !data_of) return CS_EINVAL;
    for (int32_t e = 0; e < batch; ++e) {
        if (cfg_of[e] < 0 || cfg_of[e] >= c->ncfg || data_of[e] < 0) return CS_EINVAL;
        if (c->d && data_of[e] >= c->ndata) return CS_EINVAL;
    }
    cudaDeviceSynchronize();
    free_batch(c);
    c->cfg_of.assign(cfg_of, cfg_of + batch);
    c->data_of.assign(data_of, data_of + batch);
    c->param_off.assign(batch + 1, 0);
    std::vector<int64_t> tab_off(batch);
    int64_t rows = 0, PS = 4 * (int64_t)c->maps[c->nmap].nseg;
    int32_t kmax = 0;
    for (int32_t e = 0; e < batch; ++e) {
        const CfgDev &cf = c->cfgs[cfg_of[e]];
        c->param_off[e + 1] = c->param_off[e] + cf.ktot;
        tab_off[e] = rows;
        rows += cf.K[0] + 2 * (int64_t)cf.K[1] + cf.K[2];
        PS = std::max<int64_t>(PS, (int64_t)cf.segbase[3] + c->maps[c->nmap].nseg);
        kmax = std::max(kmax, cf.ktot);
    }
    c->nparam = c->param_off[batch];
    c->nrows = rows; c->PS = PS; c->ktot_max = kmax;
    // entries grouped by configuration (stable), cut into groups of <= GROUP_MAX
    std::vector<int32_t> elist(batch);
    for (int32_t e = 0; e < batch; ++e) elist[e] = e;
    // cell-path configurations first, then the direct ones; stable inside a configuration
    auto key = [&](int32_t e) { return ((int64_t)(c->cfgs[cfg_of[e]].ncell_max > 0 ? 0 : 1) << 32) | (int64_t)cfg_of[e]; };
    std::stable_sort(elist.begin(), elist.end(), [&](int32_t a, int32_t b) { return key(a) < key(b); });
    // a group runs on the cell kernel when its configuration has a cell plan and it is long enough to amortise that
    // kernel's per-CTA set-up (plan loading, ring fill); short groups (configuration scans: one entry per
    // configuration) are ~2x faster on the direct kernel.  Cell-kernel groups come first in the array.
    std::vector<Group> groups, direct;
    for (int32_t i = 0; i < batch;) {
        int32_t j = i;
        while (j < batch && cfg_of[elist[j]] == cfg_of[elist[i]] && j - i < GROUP_MAX) ++j;
        const Group g{cfg_of[elist[i]], i, j - i, 0};
        if (c->cfgs[g.cfg].ncell_max > 0 && g.count >= c->cell_min_group) groups.push_back(g);
        else direct.push_back(g);
        i = j;
    }
    c->ngroup_cell = (int32_t)groups.size();
    groups.insert(groups.end(), direct.begin(), direct.end());
    c->ngroup = (int32_t)groups.size();
    int rc;
    std::vector<int32_t> zero_i(batch, 0);
    std::vector<Group> zero_g(batch, Group{0, 0, 0, 0});
    if ((rc = dev_upload(&c->d_cfg_of, c->cfg_of, &c->batch_bytes)) || (rc = dev_upload(&c->d_data_of, c->data_of, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_elist, elist, &c->batch_bytes)) || (rc = dev_upload(&c->d_sel_elist, zero_i, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_param_off, c->param_off, &c->batch_bytes)) || (rc = dev_upload(&c->d_tab_off, tab_off, &c->batch_bytes)) ||
        (rc = dev_upload(&c->d_groups, groups, &c->batch_bytes)) || (rc = dev_upload(&c->d_sel_groups, zero_g, &c->batch_bytes))) {
        free_batch(c);
        return rc;
    }
    const size_t tab_bytes = (size_t)rows * NROW * sizeof(float), part_bytes = (size_t)batch * PS * sizeof(double);
    if (cudaMalloc((void **)&c->d_tab, tab_bytes) != cudaSuccess || cudaMalloc((void **)&c->d_partial, part_bytes) != cudaSuccess) {
        free_batch(c);
        return CS_ENOMEM;
    }
    c->batch_bytes += (int64_t)(tab_bytes + part_bytes);
    c->batch = batch;
    return CS_OK;
}

int cs_param_offsets(cs_ctx *c, int64_t *off) {
    if (!c || c->batch <= 0 || !off) return CS_EINVAL;
    std::memcpy(off, c->param_off.data(), sizeof(int64_t) * (c->batch + 1));
    return CS_OK;
}

int cs_build_sed_tables(cs_ctx *c, const double *params, void *stream) {
    if (!c || c->batch <= 0 || !params) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    dim3 block(256);
    dim3 grid((4 * c->ktot_max + 255) / 256, std::min(c->batch, 65535));
    k_tables<<<grid, block, 0, st>>>(params, c->d_param_off, c->d_tab_off, c->d_cfg_of, c->d_cfgs, c->d_tab, c->batch, c->d_err, c->d_tc, c->skip);
    c->launches++;
    CK(cudaGetLastError());
    c->tables_built = true;
    return CS_OK;
}

static int merge_launch(cs_ctx *c, double *nll, double *grad, cudaStream_t st) {
    for (int e0 = 0; e0 < c->batch; e0 += 65535) {
        const int nb = std::min(65535, c->batch - e0);
        const int nout = (grad ? ((c->ktot_max + 31) & ~31) : 0) + 32 * c->nregion;   // virtual threads, see k_merge
        dim3 grid((nout + 255) / 256, nb);
        k_merge<<<grid, 256, 0, st>>>(c->d_partial + (int64_t)e0 * c->PS, c->PS, c->d_maps, c->d_cfgs, c->d_cfg_of + e0,
                                     c->d_param_off + e0, c->nregion, grad ? 1 : 0, nll + (int64_t)e0 * c->nregion, grad,
                                     c->skip ? c->skip + e0 : nullptr);
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
    rc = grad ? launch_like<MODE_GRAD>(c, P, 0, c->ngroup, c->ngroup_cell, st) : launch_like<MODE_VALUE>(c, P, 0, c->ngroup, c->ngroup_cell, st);
    if (rc) return rc;
    return merge_launch(c, nll, grad, st);
}

int cs_spectral_misfit(cs_ctx *c, double *chi2, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!chi2 || !c->tables_built) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LikeParams P = base_params(c);
    if ((rc = launch_like<MODE_CHI2>(c, P, 0, c->ngroup, c->ngroup_cell, st))) return rc;
    return merge_launch(c, chi2, nullptr, st);
}

int cs_component_maps(cs_ctx *c, int32_t nsel, const int32_t *entries, float *s, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!s || !c->tables_built || nsel <= 0 || nsel > c->batch) return CS_EINVAL;
    if (!entries && nsel != c->batch) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<int32_t> el(nsel);
    std::vector<Group> gr;
    gr.reserve(nsel);
    for (int32_t i = 0; i < nsel; ++i) {
        const int32_t e = entries ? entries[i] : i;
        if (e < 0 || e >= c->batch) return CS_EINVAL;
        el[i] = e;
    }
    // groups = runs of consecutive selected entries of one configuration (a group's start is its first output slot);
    // cell-path groups first
    int32_t ncell = 0;
    for (int pass = 0; pass < 2; ++pass)
        for (int32_t i = 0; i < nsel;) {
            const int32_t cf = c->cfg_of[el[i]];
            int32_t j = i;
            while (j < nsel && c->cfg_of[el[j]] == cf && j - i < GROUP_MAX) ++j;
            const bool cellp = c->cfgs[cf].ncell_max > 0 && j - i >= c->cell_min_group;
            if (cellp == (pass == 0)) {
                gr.push_back(Group{cf, i, j - i, 0});
                if (pass == 0) ++ncell;
            }
            i = j;
        }
    const int32_t ngr = (int32_t)gr.size();
    // small synchronous uploads: map output is not on the optimizer's hot path
    CK(cudaStreamSynchronize(st));
    CK(cudaMemcpy(c->d_sel_elist, el.data(), sizeof(int32_t) * nsel, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(c->d_sel_groups, gr.data(), sizeof(Group) * ngr, cudaMemcpyHostToDevice));
    LikeParams P = base_params(c);
    P.groups = c->d_sel_groups;
    P.elist = c->d_sel_elist;
    P.maps_out = s;
    return launch_like<MODE_MAPS>(c, P, 0, ngr, ncell, st);
}

int cs_cmb_variance(cs_ctx *c, double *var, void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!var || !c->tables_built) return CS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LikeParams P = base_params(c);
    if ((rc = launch_like<MODE_CMBVAR>(c, P, 0, c->ngroup, c->ngroup_cell, st))) return rc;
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
    o->ls_c1 = 1e-4; o->safe_lo = 1e-15; o->safe_hi = 1e15; o->ls_noise = 1e-6;
}

int cs_optimize(cs_ctx *c, double *params, const double *lower, const double *upper, const cs_opt *opt, double *nll_final,
                void *stream) {
    int rc = ready(c);
    if (rc) return rc;
    if (!params || !lower || !upper || !opt || opt->iters < 0 || opt->ls_max < 1 || !(opt->ls_noise >= 0) || c->batch > 65535) return CS_EINVAL;
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
    OptHyper hy{opt->lr, opt->beta1, opt->beta2, opt->eps, opt->ls_c1, opt->safe_lo, opt->safe_hi, opt->ls_noise, opt->ls_max};
    OptWork &w = c->opt;
    opt_init(w, sh, params, lower, upper, st); c->launches += 1;
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
        opt_direction(w, sh, hy, st); c->launches += 1;
        for (int ls = 0; ls < opt->ls_max; ++ls) {
            opt_trial_point(w, sh, st); c->launches += 1;
            c->skip = w.accepted;   // entries that already accepted a step sit this trial out
            r = cs_build_sed_tables(c, w.xt, st);
            if (!r) r = cs_spectral_misfit(c, w.nll_reg_t, st);
            c->skip = nullptr;
            if (r) return r;
            opt_ls_update(w, sh, hy, st); c->launches += 1;
        }
        opt_commit(w, sh, st); c->launches += 1;
        return CS_OK;
    };
    // The body is captured once into a CUDA graph and replayed: a step of a small batch is launch-bound (config 2:
    // ~30 kernels of a few microseconds each).  If the caller's stream is itself being captured, or the fused-kernel
    // timer is on, the kernels are enqueued directly.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    cudaStreamIsCapturing(st, &cap);
    bool replayed = false;
    if (opt->iters > 1 && cap == cudaStreamCaptureStatusNone && !c->prof_on) {
        if (opt->iters > 0 && (rc = iteration())) return rc;     // first iteration directly: sets function attributes, warms up
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
    int rc = cs_set_data(c, ndata, c->d_stage, ninv_host);   // the staged copy becomes the context's data
    if (rc) return rc;
    cudaStream_t cp = c->copy_stream, cm = c->comp_stream;
    // parameters and tables on the compute stream while the first data chunk is in flight on the copy stream
    CK(cudaMemcpyAsync(c->d_hparams, params_host, sizeof(double) * c->nparam, cudaMemcpyHostToDevice, cm));
    if ((rc = cs_build_sed_tables(c, c->d_hparams, cm))) return rc;
    // upload in chunks of data sets; after each chunk, launch (on the compute stream, behind an event) the groups
    // whose data are resident, so that the next chunk's copy overlaps their kernels.
    std::vector<Group> groups(c->ngroup);
    std::vector<int32_t> elist(c->batch);
    CK(cudaMemcpy(groups.data(), c->d_groups, sizeof(Group) * c->ngroup, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(elist.data(), c->d_elist, sizeof(int32_t) * c->batch, cudaMemcpyDeviceToHost));
    std::vector<int32_t> gmax(c->ngroup, 0);
    for (int g = 0; g < c->ngroup; ++g)
        for (int i = 0; i < groups[g].count; ++i) gmax[g] = std::max(gmax[g], c->data_of[elist[groups[g].start + i]]);
    std::vector<char> done(c->ngroup, 0);
    const int64_t chunk_sets = std::max<int64_t>(1, (int64_t)(128ll << 20) / (per * 4));
    LikeParams P = base_params(c);
    std::vector<cudaEvent_t> evs;
    rc = CS_OK;
    for (int64_t n0 = 0; n0 < ndata && rc == CS_OK; n0 += chunk_sets) {
        const int64_t n1 = std::min<int64_t>(ndata, n0 + chunk_sets);
        cudaEvent_t ev;
        if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { rc = CS_ECUDA; break; }
        evs.push_back(ev);
        if (cudaMemcpyAsync(c->d_stage + n0 * per, d_host + n0 * per, (size_t)((n1 - n0) * per) * sizeof(float),
                            cudaMemcpyHostToDevice, cp) != cudaSuccess ||
            cudaEventRecord(ev, cp) != cudaSuccess || cudaStreamWaitEvent(cm, ev, 0) != cudaSuccess) { rc = CS_ECUDA; break; }
        for (int g = 0; g < c->ngroup && rc == CS_OK;) {
            if (done[g] || gmax[g] >= n1) { ++g; continue; }
            int h = g;
            while (h < c->ngroup && !done[h] && gmax[h] < n1) { done[h] = 1; ++h; }
            rc = grad_host ? launch_like<MODE_GRAD>(c, P, g, h, c->ngroup_cell, cm) : launch_like<MODE_VALUE>(c, P, g, h, c->ngroup_cell, cm);
            g = h;
        }
    }
    if (rc == CS_OK) rc = merge_launch(c, c->d_hnll, grad_host ? c->d_hgrad : nullptr, cm);
    if (rc == CS_OK && cudaMemcpyAsync(nll_host, c->d_hnll, sizeof(double) * c->batch * c->nregion, cudaMemcpyDeviceToHost, cm) != cudaSuccess) rc = CS_ECUDA;
    if (rc == CS_OK && grad_host && cudaMemcpyAsync(grad_host, c->d_hgrad, sizeof(double) * c->nparam, cudaMemcpyDeviceToHost, cm) != cudaSuccess) rc = CS_ECUDA;
    if (cudaStreamSynchronize(cp) != cudaSuccess || cudaStreamSynchronize(cm) != cudaSuccess) rc = rc ? rc : CS_ECUDA;
    for (cudaEvent_t ev : evs) cudaEventDestroy(ev);
    return rc;
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
