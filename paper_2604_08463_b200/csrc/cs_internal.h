// cs_internal.h -- host/device shared declarations of libcs (not part of the public ABI).
//
// Position space.  Every configuration owns a *layout*: an order of its pixels cut into tiles of TPX positions.
//   in-place layout  position = pixel (the caller's order, HEALPix RING at the boundary); data are read from the caller's d
//   sorted layout    pixels sorted by cell = (k0, k1, k2, region), every cell padded to an even number of positions, tiles
//                    broken early when they would hold more than CELL_CAP cells; masked pixels are left out.  Every
//                    (configuration, data set) pair of the batch gets a private copy of its data in this order
//                    (k_relayout, once per cs_set_batch / cs_set_data), so that the two positions (2t, 2t+1) of a thread
//                    always share their cell and the stream of a tile is one contiguous block in HBM.
// Data layout in HBM:
//   d        [ndata][nfreq][2][npix] fp32   borrowed from the caller
//   dcopy    per sorted configuration [ntile][pairs of the configuration][2 halves][2*nfreq rows][256] fp32 ("tile-major":
//            the copies of a configuration's (cfg, data) pairs are interleaved tile by tile, so that a CTA walking the
//            entries of one tile reads one contiguous stretch -- with one copy after the other every 60-KB block of a
//            6-GB batch lay in another 2-MB page and the stream ran 6 % slower than on a 1.5-GB batch)   private
//   tab      per entry e a block of (K0 + 2*K1 + K2) rows x 16 fp32:
//              rows [0,K0)            Fd'[k][f] = cd[f] * (nu_f/nu0d)^beta_d[k]
//              rows [K0,K0+K1)        G  [k][f] = expm1(x0)/expm1(x_f),  x = h nu / (k_B T_d[k])
//              rows [K0+K1,K0+2K1)    dlnG[k][f] = d ln G / d T_d
//              rows [K0+2K1, ..+K2)   Fs'[k][f] = cs[f] * (nu_f/nu0s)^beta_s[k]
//   partial  [batch][PS] fp64   per-tile, per-segment ordered partial sums (written by the fused kernels, read by k_merge)
//            The slot of a segment inside its term's block is cluster-major (all segments of cluster 0 in ascending
//            tile order, then cluster 1, ...), so that the merge reads every cluster's partials contiguously.
//   plan     per term map in position space: idx int32[ntile*TPX], rank u16[ntile*TPX], segptr int32[ntile+1],
//            segdesc u16[nseg], segslot int32[nseg], ksegptr int32[K+1], chunkptr int32[ntile+1], segcfirst u16[nseg]
#pragma once
#include <stdint.h>

namespace cs {

constexpr int TPX = 512;       // positions per tile
constexpr int NCONS = 256;     // consumer threads of a fused kernel: thread t owns positions 2t and 2t+1 of the tile
constexpr int HALF = 256;      // a tile is staged as two halves of 256 positions (the widest TMA box)
constexpr int SEG_MAX = 32;    // longest run of ranks summed as one segment
constexpr int CHUNK_LEN = 8;   // ranks per chunk (SEG_MAX / CHUNK_LEN <= 4 chunks per segment)
constexpr int NROW = 16;       // floats per table row (nfreq padded to 16 -> 64-byte rows)
constexpr int CELL_CAP = 64;   // sorted layout: most cells per tile (a builder lane builds cells lane and lane + 32)
constexpr int CROW = 68;       // floats per cell row in shared memory: 3 columns x 16 + 16 scalars + 4 pad (= 4 mod 32 banks)
constexpr int CR_WS = 8, CR_SC = 12;    // float4 offsets of the w a_s column and of the scalars
constexpr int SC_CHUNK_CAP = 4 * (TPX / CHUNK_LEN + CELL_CAP);   // sorted layout: most chunks of the four terms of a tile
constexpr int SC_SEG_CAP = 4 * (TPX / SEG_MAX + CELL_CAP);       // and most segments
// Tile header of the sorted layout (one per configuration and tile, variable length, a multiple of 16 bytes; 32-bit words):
//   [0, HDR_META)                meta, indices HM_*
//   [HDR_META, +HDR_CONS)        per consumer thread two words: cell | r0 << 8 | r1 << 16 | r2 << 24 ; r3   (r_t = half the rank
//                                of the thread's first position in the tile's (cluster, position) order of term map t)
//   [.., + 4 ncell)              table rows (Fd', G, dlnG, Fs') of the tile's cells
//   [HM_OFF_SLOT, + nseg)        slot of every segment in the entry's partial row (terms 0..3 one after the other)
//   [HM_OFF_CDESC, ..) u16       chunk descriptors: first pair (8 bits) | (pairs-1) << 8 | term << 10
//   [HM_OFF_SDESC, ..) u16       segment descriptors: first pair | (chunks-1) << 8 | term << 10
// The loader warp of k_like_sc fetches it with one bulk copy one tile ahead of the other roles, so that a change of
// tile costs no chain of dependent global loads (a clustering scan changes tile, and configuration, with every entry).
constexpr int HDR_META = 16, HDR_CONS = 2 * NCONS;
constexpr int HM_NCELL = 0, HM_NCHUNK = 1, HM_NSEG = 2, HM_CBASE3 = 3, HM_SBASE3 = 4, HM_NSEGREG = 5, HM_SEGBASE3 = 6,
              HM_OFF_SLOT = 7, HM_OFF_CDESC = 8, HM_OFF_SDESC = 9;
constexpr int HDR_CAP_WORDS = HDR_META + HDR_CONS + 4 * CELL_CAP + SC_SEG_CAP + SC_CHUNK_CAP / 2 + SC_SEG_CAP / 2 + 4;   // longest header
constexpr int NORANK = 0xFFFF; // rank of a position that does not take part in a term's reduction

// A pivot of the LDL^T factorisation of M = A^T N^-1 A counts as non-positive (CS_ESINGULAR) when it is below this
// fraction of its diagonal entry: below it an fp32 solve carries no correct digit (R11).
constexpr float PIVOT_RTOL = 1e-6f;

constexpr int ERR_DOMAIN = 1;
constexpr int ERR_SINGULAR = 2;

// One term map (a cluster map or the region pseudo-map) in the position space of one layout.
struct MapDev {
    const int32_t *idx;       // [ntile*TPX] cluster id of the position, -1 = masked / beyond the sky
    const uint16_t *rank;     // [ntile*TPX] position in its tile's (cluster id, position) order, NORANK = none
    const int32_t *segptr;    // [ntile+1] first segment of each tile (map-local numbering)
    const uint16_t *segdesc;  // [nseg] start rank (9 bits) | (len-1) << 9
    const int32_t *segslot;   // [nseg] cluster-major slot of the segment inside its term's block of a partial row
    const int32_t *ksegptr;   // [K+1] CSR cluster -> slots [ksegptr[k], ksegptr[k+1])
    const int32_t *chunkptr;  // [ntile+1] running count of <= CHUNK_LEN-rank chunks (each segment is cut into 1..4 of them)
    const uint16_t *segcfirst;// [nseg] index of the segment's first chunk inside its tile's chunk list
    int32_t K;
    int32_t nseg;
};

// One clustering configuration: term maps for (beta_d, T_d, beta_s, region) in its layout and where each term's
// partials live.
struct CfgDev {
    int32_t map[4];       // term maps in the position space of this configuration's layout
    int32_t segbase[4];   // offset of term t inside a partial row (t = 0,1,2 gradient terms, 3 = ll / region)
    int32_t rmap[4];      // the same four maps in pixel space (in-place layout; component maps are written in pixel order)
    int32_t K[3];
    int32_t ktot;
    int32_t ntile;        // tiles of this configuration's layout
    int32_t sorted;       // 1: sorted layout with private data copies, 0: in place
    int32_t ntile_ring;   // tiles of the in-place layout
    int32_t pixbeta;      // 1: in place with beta_d (nearly) per pixel: no beta_d table rows, the direct kernel evaluates
                          //    cd (nu/nu0)^beta_d per pixel from a copy of the parameters in compensated fp32
                          //    (powerlaw_pair_f32: 2.5e-7 relative, not the bits of a table row)
    const int32_t *kseg[4];    // = maps[map[t]].ksegptr: one load less on k_merge's way to its slots
    // sorted layout only
    const uint8_t *cellid;     // [ntile*NCONS] tile-local cell of each thread (position pair)
    const int32_t *cellptr;    // [ntile+1] first cell of each tile
    const int32_t *cellrows;   // [ncell][4] table rows (Fd', G, dlnG, Fs') of the cell inside an entry's table block
    const int32_t *pospix;     // [ntile*TPX] pixel of each position, -1 = pad
    const uint32_t *hdr;       // tile headers, one after the other
    const int32_t *hdrptr;     // [ntile+1] start of each tile's header in units of 16 bytes
};

// A run of work for a fused kernel: `count` entries (elist[estart .. estart+count)) of configuration cfg on each of its
// ntile tiles = ntile*count units in (tile-major, entry-minor) order; ustart = units of the runs before this one.
struct Run {
    int32_t cfg, estart, count, ntile;
    int64_t ustart;
    const uint32_t *hdr;       // = cfgs[cfg].hdr, cfgs[cfg].hdrptr (sorted configurations; the loader's look-ahead reads
    const int32_t *hdrptr;     //   them from the run it already holds instead of chasing the configuration table)
    int64_t tstride;           // floats from one tile of a private copy to the next (sorted configurations)
};

// What the roles of a fused kernel need to know about the entry at position i of the launch's entry list, in one
// 32-byte record (two 16-byte loads) whose address does not depend on another load (a dependent global load costs a microsecond under a
// saturated HBM stream).
struct PosInfo {
    int64_t tab_row;   // first table row of the entry
    int64_t src;       // sorted configuration: float offset of the entry's private copy inside dcopy; else its data set
    int64_t param_off; // first parameter of the entry (pixbeta configurations read beta_d from the parameter copy)
    int64_t pad;
};

// Constants of the fused kernels, passed by value (constant bank).
struct KConst {
    float w[NROW];     // Ninv per band, 0 beyond nfreq
    float lnd[NROW];   // ln(nu_f/nu0d)
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
