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
//   plan     per cluster map: idx int32[npix], rank u8[ntile*TP], segptr int32[ntile+1], segdesc u16[nseg],
//            ksegptr int32[K+1], kseglist int32[nseg]
#pragma once
#include <stdint.h>

namespace cs {

constexpr int TP = 256;        // pixels per tile == threads per CTA of the fused kernel
constexpr int SEG_MAX = 32;    // longest ordered chain summed by one thread in the reduce phase
constexpr int NROW = 16;       // floats per table row (nfreq padded to 16 -> 64-byte rows)
constexpr int GROUP_MAX = 32;  // entries of one configuration handled by one CTA (per tile)

constexpr int ERR_DOMAIN = 1;
constexpr int ERR_SINGULAR = 2;

// One cluster map (or the region pseudo-map) as the kernels see it.
struct MapDev {
    const int32_t *idx;       // [npix] cluster id, -1 = masked
    const uint8_t *rank;      // [ntile*TP] position of the pixel in its tile's (cluster id, pixel) order
    const int32_t *segptr;    // [ntile+1] first segment of each tile (map-local numbering)
    const uint16_t *segdesc;  // [nseg] start (8 bits) | (len-1) << 8
    const int32_t *ksegptr;   // [K+1] CSR cluster -> segments
    const int32_t *kseglist;  // [nseg] segment ids in ascending (tile, chunk) order per cluster
    int32_t K;
    int32_t nseg;
};

// One clustering configuration: maps for (beta_d, T_d, beta_s, region) and where each term's partials live.
struct CfgDev {
    int32_t map[4];
    int32_t segbase[4];   // offset of term t inside a partial row (t = 0,1,2 gradient terms, 3 = ll / region)
    int32_t K[3];
    int32_t ktot;
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
