/*
 * kmeans_oracle.c -- plain CPU fp64 reference of spherical K-means patching (f2), written from the paper.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): nothing in the product path may call this.
 * Independent of the CUDA path and of the input generator (gen/): no shared code, headers or tables.
 *
 * The method (section 2.2): pixels are unit vectors n_p on the sphere; a patch is the set of pixels
 * nearest, in angular distance, to a centroid c_k (L100-L102) -- the smallest angle is the largest dot product n_p . c_k;
 * a Lloyd iteration replaces every centroid by the normalised mean of its pixels (L104) and assigns again.
 *
 * Readings where the paper is silent (R15).  Labels are index work and are compared bit for bit, and pixel
 * centres have symmetries that make dot products tie exactly, so every floating-point operation is fixed:
 *   dot      = (x cx + y cy) + z cz          each product and each sum rounded once (compiled with -ffp-contract=off)
 *   argmax   : a tie goes to the lowest patch id
 *   sums[k]  = pixels of patch k added one at a time in ascending pixel order
 *   centroid = sums / sqrt((sx sx + sy sy) + sz sz)    (the mean's 1/count cancels in the normalisation)
 *   a patch without pixels keeps its centroid
 * Everything below is a direct loop over that definition: no blocking, no tables, no candidate filtering.  OpenMP only
 * splits the assignment loop over pixels, whose iterations are independent.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

/* L100-L102: labels[p] = argmax_k n_p . c_k, ties to the lowest k.  vecs [n,3], cent [K,3]. */
void orc_km_assign(int64_t n, const double *vecs, int32_t K, const double *cent, int32_t *labels) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        const double x = vecs[3 * p], y = vecs[3 * p + 1], z = vecs[3 * p + 2];
        int32_t best_k = 0;
        double best = -INFINITY;
        for (int32_t k = 0; k < K; ++k) {
            const double xy = x * cent[3 * k] + y * cent[3 * k + 1];
            const double dot = xy + z * cent[3 * k + 2];
            if (dot > best) { best = dot; best_k = k; }   /* strictly greater: the first of equal maxima stays */
        }
        labels[p] = best_k;
    }
}

/* L104: c_k <- normalised mean of the pixels with labels[p] == k; an empty patch keeps c_k.  Returns 0, or -1 when
 * the work arrays cannot be allocated. */
int orc_km_update(int64_t n, const double *vecs, const int32_t *labels, int32_t K, double *cent) {
    double *sums = (double *)calloc((size_t)K * 3, sizeof(double));
    if (!sums) return -1;
    for (int64_t p = 0; p < n; ++p) {
        const int32_t k = labels[p];
        sums[3 * k] += vecs[3 * p];
        sums[3 * k + 1] += vecs[3 * p + 1];
        sums[3 * k + 2] += vecs[3 * p + 2];
    }
    for (int32_t k = 0; k < K; ++k) {
        const double sx = sums[3 * k], sy = sums[3 * k + 1], sz = sums[3 * k + 2];
        const double xx_yy = sx * sx + sy * sy;
        const double norm = sqrt(xx_yy + sz * sz);
        if (norm > 0.0) {
            cent[3 * k] = sx / norm;
            cent[3 * k + 1] = sy / norm;
            cent[3 * k + 2] = sz / norm;
        }
    }
    free(sums);
    return 0;
}

/* Sum over pixels of n_p . c_label(p): the quantity Lloyd's two steps never decrease (used by the pins). */
double orc_km_objective(int64_t n, const double *vecs, const int32_t *labels, const double *cent) {
    long double acc = 0.0L;
    for (int64_t p = 0; p < n; ++p) {
        const int32_t k = labels[p];
        acc += (long double)vecs[3 * p] * cent[3 * k] + (long double)vecs[3 * p + 1] * cent[3 * k + 1] +
               (long double)vecs[3 * p + 2] * cent[3 * k + 2];
    }
    return (double)acc;
}

/* The whole patching step: one assignment with the initial centroids (cent, in/out), then `iters` times (update,
 * assignment).  objective, when not NULL, receives [iters + 1] values of orc_km_objective, one after each assignment. */
int orc_km_lloyd(int64_t n, const double *vecs, int32_t K, double *cent, int32_t iters, int32_t *labels, double *objective) {
    orc_km_assign(n, vecs, K, cent, labels);
    if (objective) objective[0] = orc_km_objective(n, vecs, labels, cent);
    for (int32_t it = 0; it < iters; ++it) {
        if (orc_km_update(n, vecs, labels, K, cent) != 0) return -1;
        orc_km_assign(n, vecs, K, cent, labels);
        if (objective) objective[it + 1] = orc_km_objective(n, vecs, labels, cent);
    }
    return 0;
}
