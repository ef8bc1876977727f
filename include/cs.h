/*
 * cs.h -- C ABI of libcs: batched parametric spectral likelihood for CMB component separation on NVIDIA B200.
 *
 * The hot path of arxiv 2604.08463: for every batch entry e = (clustering configuration, data set,
 * parameter vector) and every unmasked pixel p
 *
 *     A_p      = [1, a_d(nu; beta_d[k0], T_d[k1]), a_s(nu; beta_s[k2])]        Eq. 2
 *     M_p      = A^T N^-1 A ,  b_S = A^T N^-1 d_S   (S = Q, U)                 L233, Eq. 5 (L76)
 *     s_S      = M^-1 b_S                                                       Eq. 5 / 8 (L76, L128)
 *     nll      = -1/2 sum_p sum_S b_S . s_S                                     Eq. 6 negated, const 0 (L80)
 *     grad[k]  = - sum_{p in k} sum_S (N^-1 (d_S - A s_S))^T (dA/dtheta_k) s_S  Eq. 17 (L241), factor 1 for this nll
 *
 * with k0,k1,k2 the pixel's cluster ids in three independent cluster maps (patch model, L93-L98).
 * Everything runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - frequencies in GHz, maps in uK_CMB, HEALPix RING order is whatever order the caller uses: the library only
 *     needs d, cluster maps and region_idx to share one pixel order.
 *   - "dev" = pointer to device memory on the current CUDA device; "host" = host memory; "any" = either (copied
 *     with cudaMemcpyDefault during the call).  Borrowed pointers must stay valid and unchanged until replaced.
 *   - every function returns CS_OK (0) or a negative CS_E* code; nothing throws; no global state (but for the fixed
 *     descriptor table of cs_spherical_kmeans_static); a context is
 *     bound to the CUDA device current at cs_create and must be used from one stream at a time.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Hot-path calls are
 *     asynchronous on it and allocate nothing.
 *
 * Parameter layout: entry e owns params[off[e] .. off[e+1]) = [beta_d x K0 ; T_d x K1 ; beta_s x K2] where
 * (K0,K1,K2) are the cluster counts of the three maps of its configuration; off[] = cs_param_offsets().
 * grad has the same layout.  nll is [batch, nregion].
 */
#ifndef CS_H
#define CS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CS_OK          0
#define CS_EINVAL     -1   /* bad argument / call order */
#define CS_EINDEX     -2   /* a cluster id or region id is out of range (checked bit-exactly, nothing computed) */
#define CS_EDOMAIN    -3   /* device error bit: T_d <= 0 or a non-finite parameter seen by cs_build_sed_tables */
#define CS_ESINGULAR  -4   /* device error bit: a pivot of the LDL^T of some pixel's M = A^T N^-1 A was not above 1e-6 of its
                              diagonal entry (covers non-positive); that entry's nll = +inf, its gradient is undefined */
#define CS_ECUDA      -5   /* a CUDA runtime call failed */
#define CS_ENOMEM     -6   /* allocation failed */
#define CS_ELIMIT     -7   /* a size is beyond the fixed capacity of an entry point that allocates nothing */

#define CS_UNITS_KCMB    0 /* dust/synchrotron columns carry the K_RJ -> K_CMB factor u(nu)/u(nu0) (default) */
#define CS_UNITS_LITERAL 1 /* Eq. 2 as printed (brightness-temperature units), no unit factor */

#define CS_MAX_NFREQ 16

/* Context options (cs_set_option).  They replace nothing in the results' meaning: every combination evaluates the same
 * sums; what changes is the pixel order in which they are streamed and reduced, hence the last bits. */
#define CS_OPT_LAYOUT        1 /* CS_LAYOUT_*; set before cs_set_clusters */
#define CS_OPT_FORM          2 /* CS_FORM_*; set before cs_set_batch */
#define CS_OPT_MIN_FILL      3 /* CS_LAYOUT_AUTO: smallest fill fraction live pixels / (tiles * 512) of a configuration's
                                  sorted layout for which it is taken (default 0.36, the measured crossover: below
                                  it, about 2.9 pixels per cell, streaming the padding costs more than the direct
                                  kernel's gathers; bench.py cellsweep); set before cs_set_clusters */
#define CS_OPT_COPY_LIMIT_MB 4 /* most device memory [MiB] the private sorted copies of a batch may take; 0 (default) =
                                  70 % of the memory free when cs_set_batch runs.  Beyond it cs_set_batch returns CS_ENOMEM. */
#define CS_OPT_PIXEL_BETA    5 /* CS_PIXBETA_*; set before cs_set_clusters */
#define CS_LAYOUT_AUTO    0 /* sorted layout for configurations whose tiles fill well, in place for the others */
#define CS_LAYOUT_INPLACE 1 /* never copy: stream the caller's d in its own pixel order (direct kernel only) */
#define CS_LAYOUT_SORTED  2 /* sorted layout for every configuration */
#define CS_FORM_AUTO      0 /* sorted-cell kernel on sorted configurations, direct kernel on the others */
#define CS_FORM_DIRECT    1 /* direct kernel everywhere, on whatever layout each configuration has (same bits) */
#define CS_PIXBETA_AUTO   0 /* a configuration that stays in place and whose beta_d map has more patches than half the
                             pixels (the paper's own optimum fits beta_d per pixel, Table 2) gets no beta_d table rows: the
                             direct kernel evaluates cd (nu/nu0)^beta_d per pixel in compensated fp32 (relative error
                             <= 2.5e-7 against 6e-8 for a table row: the last bits differ from the table path, as a
                             property of the configuration and this option, never of how entries are batched), which
                             saves 64 B written and 64 B read per pixel-eval */
#define CS_PIXBETA_OFF    1 /* always build and gather the beta_d rows */

#if defined(__GNUC__)
#define CS_API __attribute__((visibility("default")))
#else
#define CS_API
#endif

typedef struct cs_ctx cs_ctx;

/* Sky / instrument model (Eq. 2).  3 components: CMB (column of ones), dust modified black
 * body normalised at nu0_dust, synchrotron power law normalised at nu0_sync. */
typedef struct cs_model {
    int32_t nfreq;            /* 3 .. CS_MAX_NFREQ */
    const double *freqs_ghz;  /* host [nfreq] */
    double nu0_dust_ghz;      /* 353 in the paper's setup */
    double nu0_sync_ghz;      /* 23 */
    double t_cmb_k;           /* 2.7255 */
    int32_t units;            /* CS_UNITS_* */
    int64_t npix;             /* pixels per map */
} cs_model;

/* Fixed-budget optimizer options (AdaTopK, App. A, Alg. 1; hyper-parameters: DESIGN.md R13). */
typedef struct cs_opt {
    int32_t iters;      /* number of iterations (no convergence test) */
    int32_t ls_max;     /* backtracking trials per iteration (value-only evaluations) */
    double lr;          /* AdaBelief step size in [0,1] units */
    double beta1, beta2, eps;
    double ls_c1;       /* Armijo constant */
    double safe_lo, safe_hi; /* dynamic rescale range for |g_proj| (A4, L541) */
    double ls_noise;    /* Armijo slack, relative to |L|: accept when L_trial <= L + ls_c1 a min(g.d, 0) + ls_noise |L|, with
                           L = 1/2 chi^2 of the GLS residual (cs_spectral_misfit), whose fp32 evaluation noise was measured
                           at 6e-9 .. 9e-8 of itself (R13); default 1e-7; 0 = strict decrease of the computed
                           objective */
    double topk;        /* Top-K fraction in [0,1] (A2-A3, L519-L537): per iteration the max(1, floor(topk n_bound)) bound
                           parameters with the highest positive release scores are released together; 0 (default, the
                           paper's production setting, L535) releases one per iteration, 1 every one pushed inwards */
    int32_t method;     /* CS_METHOD_ADATOPK (default; Alg. 1) or CS_METHOD_LBFGS (f4(i); the L-BFGS back-end with
                           the box handled by the sigmoid reparameterisation x = l + (u - l) sigma(z); two-loop recursion over
                           `history` pairs, H0 = (s.y / y.y) I, a pair is stored when s.y > 1e-10 |s| |y|, first step and
                           fall-back -g/|g|, the same backtracking Armijo search from alpha = 1 on 1/2 chi^2 (ls_c1, ls_max,
                           ls_noise); a start on a bound is moved to 1e-6 of the width inside; lr, beta*, eps, safe_*, topk
                           are not used; R19) */
    int32_t history;    /* L-BFGS pairs kept, 1 .. 32 (default 10) */
} cs_opt;
#define CS_METHOD_ADATOPK 0
#define CS_METHOD_LBFGS 1

/* Create a context for `model`.  Allocates only small constant tables.  *out is NULL on failure. */
CS_API int cs_create(cs_ctx **out, const cs_model *model);
CS_API int cs_destroy(cs_ctx *ctx);

/* Sets a context option (CS_OPT_*).  CS_EINVAL for an unknown key, a bad value, or a call after the step that reads it. */
CS_API int cs_set_option(cs_ctx *ctx, int32_t key, double value);

/* Patch model: `maps` holds nmap cluster maps [nmap, npix] int32 (any); Kmap[nmap] (host) their
 * cluster counts; a clustering configuration c is a triple cfg_maps[c] = (map for beta_d, map for T_d, map for
 * beta_s) (host [ncfg,3]).  A cluster id of -1 in any of a configuration's three maps masks the pixel for that
 * configuration (L211).  region_idx (any, [npix], values < nregion) or NULL with nregion = 1 splits nll by sky
 * region (L269).  Validates -1 <= id < K bit-exactly (CS_EINDEX otherwise, context unchanged), copies the maps
 * (the caller may free them) and builds the per-tile segment plan of the ordered cluster reduction and, per
 * configuration, its layout (CS_OPT_LAYOUT): in place, or sorted by cell = (k0, k1, k2, region) with cells padded to an
 * even number of positions, for which every (configuration, data set) pair of a batch later gets a private copy of
 * its data (cs_set_batch / cs_set_data), streamed by the sorted-cell kernel.  Which kernel runs is a property of the
 * configuration and the options, never of how entries are grouped into batches. */
CS_API int cs_set_clusters(cs_ctx *ctx, int32_t nmap, const int32_t *maps, const int32_t *Kmap,
                    int32_t ncfg, const int32_t *cfg_maps, const uint8_t *region_idx, int32_t nregion);

/* Layout taken for configuration cfg: *sorted = 1 / 0, *ntile = its 512-position tiles, *fill = live pixels / (ntile * 512)
 * (any output may be NULL). */
CS_API int cs_layout_info(cs_ctx *ctx, int32_t cfg, int32_t *sorted, int32_t *ntile, double *fill);

/* Data (Eq. 1): d dev [ndata, nfreq, 2, npix] fp32 (Q then U per band, pixel fastest), borrowed;
 * ninv any [nfreq] fp32 = 1/sigma_f^2, the same for Q, U and every pixel (L219), copied.  When a batch is set, the
 * private copies of its sorted configurations are gathered here (synchronous): call again after changing d in place.
 * A data_of beyond ndata in the current batch gives CS_EINVAL and leaves the context unchanged. */
CS_API int cs_set_data(cs_ctx *ctx, int32_t ndata, const float *d, const float *ninv);

/* Batch: entry e evaluates configuration cfg_of[e] on data set data_of[e] (both host [batch]).  Allocates the
 * SED tables, the reduction workspace and the private sorted copies for this batch (the only allocation outside
 * cs_create/cs_set_clusters) and, when the data are set, gathers the copies (synchronous).
 * Memory: every distinct (sorted configuration, data set) pair of the batch holds one private copy of
 * ntile x 512 positions x nfreq x 2 x 4 B (ntile from cs_layout_info: 61440 B a tile at nfreq 15; 6.0 MB a pair at
 * nside 64 with well filled tiles, 1 / fill times the data otherwise), within CS_OPT_COPY_LIMIT_MB, else CS_ENOMEM with
 * the context left as after cs_set_clusters.  A job larger than that -- the paper's 13,824 configurations x 40
 * realisations on three regions is 552,960 pairs = 3.5 TB of copies -- is walked by the caller in
 * batches: keep the 40 data sets resident (cs_set_data once), and per batch call cs_set_clusters with a slice of the
 * configurations (about 500 of them x 40 realisations = 20,000 pairs fill 70 % of a 180-GB B200) and cs_set_batch;
 * configurations never interact, so results do not depend on the slicing. */
CS_API int cs_set_batch(cs_ctx *ctx, int32_t batch, const int32_t *cfg_of, const int32_t *data_of);

/* off host [batch+1] int64: parameter offsets of the current batch. */
CS_API int cs_param_offsets(cs_ctx *ctx, int64_t *off);

/* a1 (Eq. 2): per entry, cluster and band the separable SED factors cd*(nu/nu0d)^beta_d, the Planck ratio
 * B-factor G(nu,T_d), its log-derivative dlnG/dT_d and cs*(nu/nu0s)^beta_s, evaluated in fp64 and stored fp32.
 * params dev fp64 (layout above).  Sets the sticky device bit CS_EDOMAIN on T_d <= 0 / non-finite input.
 * The later calls read the tables, not `params`: the caller may overwrite them (in stream order) after the call.  For a
 * configuration that stays in place with beta_d (nearly) per pixel (CS_OPT_PIXEL_BETA) the beta_d rows are not built;
 * the fused kernel evaluates them per pixel from a copy of `params` that the library makes on `stream` when the batch
 * holds such a configuration (relative error <= 2.5e-7 instead of 6e-8; same tolerances). */
CS_API int cs_build_sed_tables(cs_ctx *ctx, const double *params, void *stream);

/* a2+a3: fused per-pixel likelihood / gradient and the ordered fp64 reduction onto clusters, for the tables last
 * built.  nll dev [batch*nregion] fp64; grad dev fp64 (parameter layout) or NULL for value only.
 * Results are bitwise reproducible and independent of how entries are grouped into batches. */
CS_API int cs_spectral_like_grad(cs_ctx *ctx, double *nll, double *grad, void *stream);

/* chi^2 of the GLS residual per entry and region, chi2 dev [batch*nregion] fp64:
 *     chi2 = sum_p sum_S sum_f Ninv_f (d_S - A s_S)_f^2  =  2 nll + d^T N^-1 d            (Eq. 3 at the GLS solution, L66)
 * for the tables last built.  It differs from 2 nll by a parameter-independent constant but is evaluated from the
 * residual itself, so small changes of the objective are resolved (nll = -1/2 b.s carries the fp32 rounding of a number
 * ~1e5 times larger); cs_optimize runs its line search on it. */
CS_API int cs_spectral_misfit(cs_ctx *ctx, double *chi2, void *stream);

/* a4 (Eq. 5/8): GLS component maps s dev [nsel, 3, 2, npix] fp32 (cmb, dust@nu0d, sync@nu0s; Q,U) for entries
 * `entries` (host [nsel], read during the call) or all entries in order when entries == NULL (then nsel must equal
 * batch).  Masked pixels are written as 0.  Asynchronous on `stream` like the other hot-path calls (the selection
 * travels through a pinned staging ring; nothing is allocated and the stream is not synchronised). */
CS_API int cs_component_maps(cs_ctx *ctx, int32_t nsel, const int32_t *entries, float *s, void *stream);

/* Map level of the residual estimates of Eq. 14-15: cmb dev [nsel, 2, npix] fp32 =
 * [W_e d_j]_CMB, the CMB row (Q, U) of the map-making operator W = (A^T N^-1 A)^-1 A^T N^-1 of entry entries[i]
 * (its configuration and the parameters the tables were last built with) applied to data set j = data_sel[i] of the
 * current data -- any data set, not only the entry's own.  With d_j the noise-free foreground-only maps d_fg it is
 * the systematic residual [W d_fg]_CMB of Eq. 15; the statistical residual of Eq. 14 is the caller's difference
 * (s_hat_CMB - s_CMB^true) - [W d_fg]_CMB.  entries == NULL takes all entries in order; data_sel host [nsel], required.
 * Masked pixels are written as 0.  Asynchronous like cs_component_maps.  (The spectra C_l of those maps are out of
 * scope: they need spherical-harmonic transforms.) */
CS_API int cs_cmb_residual_maps(cs_ctx *ctx, int32_t nsel, const int32_t *entries, const int32_t *data_sel, float *cmb, void *stream);

/* f3, the cell-compressed likelihood (PAPER.md:L95 patch model, L80 Eq. 6): pixels with the same cluster triple share
 * A, so their part of Eq. 6 is tr(M^-1 A^T T A) with the parameter-independent second moments
 * T = N^-1 (sum_{p,S} d_S d_S^T) N^-1 of the cell.  cs_cell_moments builds T (fp64, on the fp64 tensor cores, from the pair's private sorted copy) for every (configuration, data set)
 * pair of the current batch from the current data -- call it once after cs_set_data / cs_set_batch, and again when the
 * data change; it allocates its workspace on the first call.  cs_spectral_like_grad_cells then evaluates nll and grad
 * (same meaning, layout and tolerances as cs_spectral_like_grad) for the tables last built, from T alone, in fp64: one
 * 15 x 15 contraction per cell instead of one pass over every pixel.  It pays when cells hold more than ~8 pixels
 * (a clustering scan over coarse configurations) and is slower than the per-pixel path at K ~ npix.
 * Requirements: nfreq <= 15 and every configuration of the batch on the sorted layout (CS_EINVAL otherwise). */
CS_API int cs_cell_moments(cs_ctx *ctx, void *stream);
CS_API int cs_spectral_like_grad_cells(cs_ctx *ctx, double *nll, double *grad, void *stream);

/* f1 (Eq. 10): per entry and region, variance over unmasked pixels of the reconstructed CMB map, Q and U
 * summed: var dev [batch*nregion] fp64, computed without writing the maps. */
CS_API int cs_cmb_variance(cs_ctx *ctx, double *var, void *stream);

/* a5: device-resident fixed-budget optimizer -- AdaTopK (Alg. 1) or, with opt->method = CS_METHOD_LBFGS, L-BFGS -- on
 * every entry independently.  It calls cs_build_sed_tables,
 * cs_spectral_like_grad (value + gradient, once per iteration) and cs_spectral_misfit (the objective of the line-search
 * trials: 1/2 chi^2 = nll + const, R13 -- a deviation from north_star's "only the first two").
 * params dev in: start, out: result; lower/upper dev, same layout; nll_final dev [batch] (summed over regions) or
 * NULL.  Any batch size (the per-entry kernels put the entry on grid.x).  No host synchronisation.  The iteration body is captured
 * into a CUDA graph and replayed unless `stream` is itself being captured; on the legacy default stream the work is
 * forked onto an internal stream and joined back before the call returns (still asynchronous to the host).
 * Line-search trials skip the entries that have already accepted a step. */
CS_API int cs_optimize(cs_ctx *ctx, double *params, const double *lower, const double *upper, const cs_opt *opt,
                double *nll_final, void *stream);
CS_API void cs_opt_defaults(cs_opt *opt);

/* Convenience for end-to-end use from host memory: uploads d_host [ndata,nfreq,2,npix] (pinned or pageable) in
 * chunks overlapped with compute, evaluates the current batch and returns nll / grad in host memory.
 * Requires data_of to be non-decreasing over the batch.  Synchronous. */
CS_API int cs_eval_host(cs_ctx *ctx, int32_t ndata, const float *d_host, const float *ninv_host, const double *params_host,
                 double *nll_host, double *grad_host);

/* f2, batched spherical K-means patching, the step before the path; needs no context.
 * nprob independent problems on the same pixel set: vecs dev [npix,3] fp64 unit vectors of the pixel centres; problem j
 * has K[j] patches (host [nprob]) and, when prob_region != NULL and prob_region[j] >= 0, only the pixels with
 * region[p] == prob_region[j] (region dev [npix] uint8) take part.  cent dev [sum_j K[j], 3] fp64: in = the initial
 * centroids (the caller draws them), out = the final ones.  Runs one assignment, then `iters` Lloyd iterations
 * (centroid = renormalised mean of its pixels, an empty patch keeps its centroid; assignment = largest dot product in
 * fp64, ties to the lowest id).  labels dev [nprob, npix] int32: patch id in [0, K[j]), or -1 outside the problem's
 * region.  The arithmetic is fixed operation by operation (csrc/cs_kmeans.cuh), so labels are reproducible bit for
 * bit.  Asynchronous on `stream`. */
CS_API int cs_spherical_kmeans(int64_t npix, const double *vecs, const uint8_t *region, int32_t nprob, const int32_t *K,
                        const int32_t *prob_region, double *cent, int32_t iters, int32_t *labels, void *stream);

/* cs_spherical_kmeans for callers that must not allocate device memory.
 *
 * Who needs it: a host program that has given all of device memory to a pool of its own (an inference server, a
 * framework allocator with a hard cap), so that a cudaMalloc from inside a library can fail at any moment; and a
 * latency-bound loop that cannot take the device-wide synchronisation an allocation or a free may bring.
 * cs_spherical_kmeans keeps its per-problem descriptors (patch count, region, centroid offset: 16 bytes a problem) in a
 * table it allocates and frees on every call.  This entry point runs the same two kernels on the same inputs and gives
 * the same bits in `cent` and `labels`, but keeps that table in a fixed array that is part of the library image:
 * CS_KMEANS_STATIC_MAX_PROB descriptors = 16 KiB, held by every GPU that loads libcs.so until the process exits.
 * It calls no cudaMalloc, cudaFree, stream-ordered allocator or other allocating routine, on the device or the host;
 * inputs and outputs are the caller's, with the layouts of cs_spherical_kmeans.
 *
 *   - nprob > CS_KMEANS_STATIC_MAX_PROB returns CS_ELIMIT and launches nothing; split the problems over several calls.
 *   - The first call on each device looks up the device address of the table (cudaGetSymbolAddress, with that device
 *     current, result checked and remembered per device).  Make that first call outside any stream capture.
 *   - One table serves every call on a device and keeps what the last call wrote.  Nothing in it has to start at zero:
 *     a call overwrites the nprob descriptors it will read, in stream order, before its first kernel, and reads no others.
 *     Calls issued to the same stream therefore queue up correctly.  Calls that can overlap on the GPU (different streams
 *     without an event between them, or different host threads doing so) race on the table: serialise them. */
#define CS_KMEANS_STATIC_MAX_PROB 1024
CS_API int cs_spherical_kmeans_static(int64_t npix, const double *vecs, const uint8_t *region, int32_t nprob, const int32_t *K,
                               const int32_t *prob_region, double *cent, int32_t iters, int32_t *labels, void *stream);

/* Synchronises `stream`, returns and clears the sticky device error bits: CS_OK, CS_EDOMAIN or CS_ESINGULAR. */
CS_API int cs_check(cs_ctx *ctx, void *stream);
CS_API const char *cs_strerror(int code);

/* Optional device timing of the fused kernel: when enabled, every gradient-mode launch of the fused per-pixel kernel
 * is bracketed by CUDA events on its own stream (ring of 512 launches).  cs_profile_read synchronises the device and
 * returns the summed duration [ms] and the number of launches measured since cs_profile(ctx, 1). */
CS_API int cs_profile(cs_ctx *ctx, int enable);
CS_API int cs_profile_read(cs_ctx *ctx, double *total_ms, int64_t *count);

/* The parameter-independent constants the table and fused kernels are given, computed on the host once per context
 * (cs_create) or data set (cs_set_data); any output may be NULL.  Host [nfreq] each:
 *   cd[f]  = (nu_f/nu0d) u(nu_f)/u(nu0d)   dust band constant: (nu/nu0)^(beta_d+1) = (nu/nu0) (nu/nu0)^beta_d times the
 *                                           K_RJ -> K_CMB factor u = (e^x-1)^2 / (x^2 e^x), x = h nu / (k T_cmb)   (Eq. 2, R1-R2)
 *   cs[f]  = u(nu_f)/u(nu0s)               synchrotron band constant (1 in CS_UNITS_LITERAL, like the u ratio of cd)
 *   lnd[f] = ln(nu_f/nu0d), lns[f] = ln(nu_f/nu0s)   the log-derivatives of the two power laws
 *   *inv_sum_w = 1 / sum_f Ninv_f (fp32 as the kernels use it; 0 before cs_set_data).
 * For tests: they are compared with the oracle's own evaluation of the same expressions. */
CS_API int cs_model_constants(cs_ctx *ctx, double *cd, double *cs, double *lnd, double *lns, double *inv_sum_w);

/* Introspection used by the bench and the tests. */
CS_API int64_t cs_workspace_bytes(cs_ctx *ctx);      /* device bytes currently held by the context */
CS_API int64_t cs_kernel_launches(cs_ctx *ctx);      /* kernels launched by this context so far */
CS_API int cs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CS_H */
