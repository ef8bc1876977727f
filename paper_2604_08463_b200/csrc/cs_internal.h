// cs_internal.h -- host/device shared declarations of libcs (not part of the public ABI).
//
// Data layout in HBM:
//   d        [ndata][nfreq][2][npix] fp32   borrowed from the caller, streamed once per pixel-eval
//   tab      per entry e a block of (K0 + 2*K1 + K2) rows x 16 fp32:
//              rows [0,K0)            Fd'[k][f] = cd[f] * (nu_f/nu0d)^beta_d[k]
//              rows [K0,K0+K1)        G  [k][f] = expm1(x0)/expm1(x_f),  x = h nu / (k_B T_d[k])
//              rows [K0+K1,K0+2K1)    dlnG[k][f] = d ln G / d T_d
//              rows [K0+2K1, ..+K2)   Fs'[k][f] = cs[f] * (nu_f/nu0s)^beta_s[k]
//   partial  [batch][PS] fp64   per-tile, per-segment ordered partial sums (written by k_like, read by k_merge)
//            The slot of a segment inside its term's block is cluster-major (all segments of cluster 0 in ascending
//            tile order, then cluster 1, ...), so that the merge reads every cluster's partials contiguously.
//   plan     per cluster map: idx int32[npix], rank u8[ntile*TP], segptr int32[ntile+1], segdesc u16[nseg],
//            segslot int32[nseg], ksegptr int32[K+1]
//   cells    per clustering configuration (cell path only): the distinct (k0,k1,k2) triples of every tile in order of
//            first appearance: cellid u8[ntile*TP] (0xFF = masked pixel), cellptr int32[ntile+1],
//            rowlist int32[nrow] = the distinct table rows a tile's cells read (rowptr int32[ntile+1]),
//            cellrows int32[ncell][4] = slots of the cell's rows (Fd', G, dlnG, Fs') in its tile's row list
#pragma once
#include <stdint.h>

namespace cs {

constexpr int TP = 256;        // pixels per tile == threads per CTA of the fused kernel
constexpr int SEG_MAX = 32;    // longest ordered chain summed by one thread in the reduce phase
constexpr int NROW = 16;       // floats per table row (nfreq padded to 16 -> 64-byte rows)
constexpr int GROUP_MAX = 64;  // entries of one configuration handled by one CTA (per tile)
constexpr int CELL_MIN_GROUP = 12;   // shortest group (entries of one configuration) worth the cell kernel's set-up
constexpr int CELL_CAP = 96;   // cell path: most distinct cluster triples a tile may hold (else the direct kernel runs)
constexpr int CHUNK_LEN = 8;   // cell kernel reduce: ranks summed by one lane in one step (SEG_MAX / CHUNK_LEN <= 4)
constexpr int CHUNK_CAP = 416; // cell kernel reduce: most chunks (and segments) of the four terms of one tile
constexpr int ROW_CAP = 128;   // cell path: most distinct table rows the cells of one tile may read
constexpr int CSTRIDE = 36;    // floats per cell row in shared memory: 16 column values + 16 scalars + 4 pad (= 4 mod 32 banks)

// A pivot of the LDL^T factorisation of M = A^T N^-1 A counts as non-positive (CS_ESINGULAR) when it is below this
// fraction of its diagonal entry: below it an fp32 solve carries no correct digit (R11).
constexpr float PIVOT_RTOL = 1e-6f;

constexpr int ERR_DOMAIN = 1;
constexpr int ERR_SINGULAR = 2;

// One cluster map (or the region pseudo-map) as the kernels see it.
struct MapDev {
    const int32_t *idx;       // [npix] cluster id, -1 = masked
    const uint8_t *rank;      // [ntile*TP] position of the pixel in its tile's (cluster id, pixel) order
    const int32_t *segptr;    // [ntile+1] first segment of each tile (map-local numbering)
    const uint16_t *segdesc;  // [nseg] start (8 bits) | (len-1) << 8
    const int32_t *segslot;   // [nseg] cluster-major slot of the segment inside its term's block of a partial row
    const int32_t *ksegptr;   // [K+1] CSR cluster -> slots [ksegptr[k], ksegptr[k+1])
    const int32_t *chunkptr;  // [ntile+1] running count of <= CHUNK_LEN-rank chunks (each segment is cut into 1..4 of them)
    const uint16_t *segcfirst;// [nseg] index of the segment's first chunk inside its tile's chunk list
    int32_t K;
    int32_t nseg;
};

// One clustering configuration: maps for (beta_d, T_d, beta_s, region) and where each term's partials live.
struct CfgDev {
    int32_t map[4];
    int32_t segbase[4];   // offset of term t inside a partial row (t = 0,1,2 gradient terms, 3 = ll / region)
    int32_t K[3];
    int32_t ktot;
    // cell plan (null / 0 when the configuration runs on the direct kernel)
    const uint8_t *cellid;     // [ntile*TP]
    const int32_t *cellptr;    // [ntile+1]
    const int32_t *cellrows;   // [ncell][4] tile-local row slots (Fd', G, dlnG, Fs') into the tile's row list
    const int32_t *rowptr;     // [ntile+1]
    const int32_t *rowlist;    // [nrow] distinct table rows (of an entry's table block) the tile's cells read
    int32_t ncell_max;         // most cells in one tile; 0 = direct path
    int32_t pad;
};

struct Group {
    int32_t cfg;
    int32_t start;   // into elist
    int32_t count;
    int32_t pad;
};

// Constants of the fused kernel, passed by value (constant bank).
struct KConst {
    float w[NROW];     // Ninv per band, 0 beyond nfreq
    float lnd[NROW];   // ln(nu_f/nu0d)
    float lnsw[NROW];  // ln(nu_f/nu0s) * w_f
    float lns[NROW];   // ln(nu_f/nu0s)
    float invw[NROW];  // 1 / w_f (0 beyond nfreq)
    float inv_m00;     // 1 / sum_f w_f
    float m00;
};

// Constants of the table kernel (fp64).
struct TConst {
    double cd[NROW], cs[NROW], lnd[NROW], lns[NROW], nu[NROW];
    double nu0d, hk;   // hk = h*1e9/k_B [K/GHz]
    int32_t nfreq;
};

}  // namespace cs
