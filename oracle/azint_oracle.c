/*
 * azint_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the 1D azimuthal-integration hot path computes:
 * bounding-box pixel splitting as a FORWARD scatter ("loops over all the pixels of the detector, adding their
 * contributions to the appropriate bins", section 4.1), followed by the ratio of the weighted and
 * unweighted histograms (section 3.3).  The CUDA path reaches the same sums in another
 * order (gather / sparse matrix), so this file is the definition it is checked against.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this library.
 * It shares no code with paper_1412_6367_b200/csrc and includes none of its headers.
 *
 * Steps (notation of DESIGN.md section 3, which restates SURVEY.md section 8(c) O1-O7):
 *   O1  radial extent [r_min, r_max] of the pixel rectangle   (PAPER.md:50 r = sqrt((x-xc)^2+(y-yc)^2)
 *       "rectangular box circumscribing the actual pixel")
 *   O2  unit transform u(r): r, 2theta = atan(r/d), q = 4 pi sin(2theta/2)/lambda
 *   O3  bins: npt equal-width bins on [u0, u1]; default range = extent of all pixels
 *   O4  split: outermost bins get their fractional overlap, internal bins share the rest evenly
 *   O5  per-pixel value v = (I - dark) / (flat * solidangle * polarization)
 *   O6  S[b] += c v,  C[b] += c
 *   O7  intensity = S / C
 *
 * Parity pins (tests/test_oracle_pins.py): hand-worked split, the 2x2 worked example, mpmath brute force of every
 * coefficient on tiny images, closed-form ranges, conservation of signal and of pixel count, uniform
 * image, npt = 1 mean, scipy CSR product, Bragg ring positions, the nnz / row-length statistics of
 * SURVEY.md section 8(a).  The bidimensional routines at the end of the file are pinned in tests/test_oracle_pins_2d.py:
 * the sum over the azimuthal bins equals the (pinned) 1D result bin by bin, per-pixel weights sum to 1, conservation,
 * a hand-worked 2x2 image, 4-fold symmetry, mpmath brute force of the azimuthal extents (seam, centre inside / on an
 * edge / on a corner).  Non-finite inputs (a NaN / Inf pixel, dark current or denominator = an invalid pixel, DESIGN.md
 * reading 8) are pinned as "exactly the result of masking that pixel" (tests/test_oracle_pins.py); <= 1 ulp bin-edge ties
 * are reported, not asserted.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).  No fast-math; IEEE double throughout.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double distance_m, pixel_y_m, pixel_x_m, center_y_px, center_x_px, wavelength_m;
} aio_geometry;

enum { AIO_R_MM = 0, AIO_TTH_DEG = 1, AIO_TTH_RAD = 2, AIO_Q_NM = 3, AIO_Q_A = 4 };

static double max3(double a, double b, double c) { double m = a > b ? a : b; return m > c ? m : c; }
static double max2(double a, double b) { return a > b ? a : b; }
static double min2(double a, double b) { return a < b ? a : b; }

/* O2: radial coordinate in the requested unit, r in metres. */
static double unit_of_r(double r, const aio_geometry *g, int unit)
{
    const double pi = 3.14159265358979323846;
    switch (unit) {
    case AIO_R_MM:    return 1e3 * r;
    case AIO_TTH_RAD: return atan(r / g->distance_m);
    case AIO_TTH_DEG: return atan(r / g->distance_m) * 180.0 / pi;
    case AIO_Q_NM:    return 1e-9 * (4.0 * pi * sin(atan(r / g->distance_m) / 2.0) / g->wavelength_m);
    case AIO_Q_A:     return 1e-10 * (4.0 * pi * sin(atan(r / g->distance_m) / 2.0) / g->wavelength_m);
    }
    return NAN;
}

/* O1 + O2 for pixel (i, j): the pixel occupies [j, j+1] x [i, i+1] in pixel units. */
static void pixel_bounds(const aio_geometry *g, int unit, int i, int j, double *u_min, double *u_max)
{
    double x_lo = ((double)j - g->center_x_px) * g->pixel_x_m;
    double x_hi = ((double)(j + 1) - g->center_x_px) * g->pixel_x_m;
    double y_lo = ((double)i - g->center_y_px) * g->pixel_y_m;
    double y_hi = ((double)(i + 1) - g->center_y_px) * g->pixel_y_m;
    /* nearest point of the rectangle to the beam centre (0 along an axis the centre projects inside of) */
    double nx = max3(x_lo, -x_hi, 0.0);
    double ny = max3(y_lo, -y_hi, 0.0);
    /* farthest corner */
    double fx = max2(fabs(x_lo), fabs(x_hi));
    double fy = max2(fabs(y_lo), fabs(y_hi));
    double r_min = sqrt(nx * nx + ny * ny);
    double r_max = sqrt(fx * fx + fy * fy);
    *u_min = unit_of_r(r_min, g, unit);
    *u_max = unit_of_r(r_max, g, unit);
}

int aio_pixel_bounds(const aio_geometry *g, int height, int width, int unit, double *u_min, double *u_max)
{
    if (!g || height < 1 || width < 1 || unit < 0 || unit > 4) return -1;
    for (int i = 0; i < height; ++i)
        for (int j = 0; j < width; ++j)
            pixel_bounds(g, unit, i, j, &u_min[(int64_t)i * width + j], &u_max[(int64_t)i * width + j]);
    return 0;
}

/* O3: automatic range = [min u_min, max u_max] over ALL pixels (independent of any mask). */
int aio_auto_range(const double *u_min, const double *u_max, int64_t n, double *u0, double *u1)
{
    if (n < 1) return -1;
    double lo = u_min[0], hi = u_max[0];
    for (int64_t p = 1; p < n; ++p) {
        if (u_min[p] < lo) lo = u_min[p];
        if (u_max[p] > hi) hi = u_max[p];
    }
    *u0 = lo; *u1 = hi;
    return 0;
}

/*
 * O4 for one pixel.  In bin units f = (u - u0)/delta the pixel covers [f_min, f_max]; bin b is [b, b+1), the last bin
 * closed.  Writes up to `cap` (bin, coefficient) pairs and returns how many the pixel has (may exceed cap).
 *   whole pixel in one bin        -> coefficient 1                         ("no pixel splitting")
 *   left / right outermost bins   -> (b_min+1-f_min)/w and (f_max-b_max)/w ("calculated first")
 *   internal bins                 -> 1/w each                              ("evenly distributed")
 * all of which is  overlap([f_min,f_max], [b,b+1]) / (f_max - f_min).
 */
int aio_split(double u_min, double u_max, double u0, double u1, int npt, int *bins, double *coefs, int cap)
{
    double delta = (u1 - u0) / (double)npt;
    double f_min = (u_min - u0) / delta;
    double f_max = (u_max - u0) / delta;
    double w = f_max - f_min;
    int n = 0;
    if (!(f_max > 0.0) || !(f_min < (double)npt)) return 0;       /* entirely outside the range */
    if (!(w > 0.0)) {                                               /* degenerate zero-width pixel */
        int b = (int)floor(f_min);
        if (b > npt - 1) b = npt - 1;
        if (b < 0) b = 0;
        if (cap > 0) { bins[0] = b; coefs[0] = 1.0; }
        return 1;
    }
    double a = max2(f_min, 0.0);
    double z = min2(f_max, (double)npt);
    int b_first = (int)floor(a);
    int b_last = (int)floor(z);
    if (b_last > npt - 1) b_last = npt - 1;
    for (int b = b_first; b <= b_last; ++b) {
        double ov = min2(z, (double)(b + 1)) - max2(a, (double)b);
        if (ov > 0.0) {
            if (n < cap) { bins[n] = b; coefs[n] = ov / w; }
            ++n;
        }
    }
    return n;
}

#define AIO_MAX_SPLIT 4096

/* O5: corrected value and validity of one pixel. */
static int pixel_value(int64_t p, const double *image, const double *dark, const double *flat,
                       const double *solidangle, const double *polarization, const uint8_t *mask, double *v)
{
    if (mask && mask[p]) return 0;
    double den = 1.0;
    if (flat) den *= flat[p];
    if (solidangle) den *= solidangle[p];
    if (polarization) den *= polarization[p];
    double num = image[p] - (dark ? dark[p] : 0.0);
    if (den == 0.0 || !isfinite(den) || !isfinite(num)) return 0;
    *v = num / den;
    return 1;
}

/*
 * O4-O7 as a forward scatter over precomputed pixel bounds (one frame).  This is also the routine bench.py times as the
 * CPU baseline ("per-frame integrate"): bounds are geometry-only and computed once per detector, as in the paper.
 * nthreads > 1 uses the paper's own multi-thread scheme: image rows split across threads, one private pair of
 * histograms per thread, merged at the end (section 3.4.1).  nthreads = 1 is the parity reference.
 */
int aio_integrate1d_bounds(const double *u_min, const double *u_max, int64_t npix, int npt, double u0, double u1,
                           const double *image, const double *dark, const double *flat, const double *solidangle,
                           const double *polarization, const uint8_t *mask, double empty_value, int nthreads,
                           double *radial, double *intensity, double *sum_signal, double *count)
{
    if (npix < 1 || npt < 1 || !(u1 > u0) || !image) return -1;
    if (nthreads < 1) nthreads = 1;
    double delta = (u1 - u0) / (double)npt;
    double *S = (double *)calloc((size_t)nthreads * npt, sizeof(double));
    double *C = (double *)calloc((size_t)nthreads * npt, sizeof(double));
    if (!S || !C) { free(S); free(C); return -2; }
    int overflow = 0;      /* a pixel that spans more than AIO_MAX_SPLIT bins is an error here as in aio_csr (-3) */
#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads)
#endif
    {
        int t = 0, nt = 1;
#ifdef _OPENMP
        t = omp_get_thread_num(); nt = omp_get_num_threads();
#endif
        double *St = S + (size_t)t * npt, *Ct = C + (size_t)t * npt;
        int64_t lo = npix * t / nt, hi = npix * (t + 1) / nt;
        int bins[AIO_MAX_SPLIT]; double coefs[AIO_MAX_SPLIT];
        for (int64_t p = lo; p < hi; ++p) {
            double v;
            if (!pixel_value(p, image, dark, flat, solidangle, polarization, mask, &v)) continue;
            int n = aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
            if (n > AIO_MAX_SPLIT) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
                overflow = 1;
                continue;
            }
            for (int k = 0; k < n; ++k) {
                St[bins[k]] += coefs[k] * v;      /* weighted histogram   */
                Ct[bins[k]] += coefs[k];          /* unweighted histogram */
            }
        }
    }
    if (overflow) { free(S); free(C); return -3; }
    for (int t = 1; t < nthreads; ++t)
        for (int b = 0; b < npt; ++b) { S[b] += S[(size_t)t * npt + b]; C[b] += C[(size_t)t * npt + b]; }
    for (int b = 0; b < npt; ++b) {
        if (radial) radial[b] = u0 + ((double)b + 0.5) * delta;
        sum_signal[b] = S[b];
        count[b] = C[b];
        intensity[b] = C[b] > 0.0 ? S[b] / C[b] : empty_value;
    }
    free(S); free(C);
    return 0;
}

/*
 * The other estimator (SURVEY.md section 8(c) reading 9, "summed normalisation"): instead of correcting every pixel and
 * averaging, sum the dark-subtracted signal and the normalisation separately with the same weights and divide the sums:
 *   sum_signal[b] = sum c (I - dark),   sum_norm[b] = sum c (flat * solidangle * polarization),
 *   intensity[b] = sum_signal[b] / sum_norm[b]   (empty_value where sum_norm[b] == 0).
 * Validity of a pixel is O5's.  The paper lists the corrections but not where the division happens; this
 * variant is an option of the library (ai_set_normalization), the default stays O5-O7 above.
 */
int aio_integrate1d_bounds_split(const double *u_min, const double *u_max, int64_t npix, int npt, double u0, double u1,
                                 const double *image, const double *dark, const double *flat, const double *solidangle,
                                 const double *polarization, const uint8_t *mask, double empty_value,
                                 double *intensity, double *sum_signal, double *sum_norm)
{
    if (npix < 1 || npt < 1 || !(u1 > u0) || !image) return -1;
    int bins[AIO_MAX_SPLIT]; double coefs[AIO_MAX_SPLIT];
    for (int b = 0; b < npt; ++b) { sum_signal[b] = 0.0; sum_norm[b] = 0.0; }
    for (int64_t p = 0; p < npix; ++p) {
        double v;
        if (!pixel_value(p, image, dark, flat, solidangle, polarization, mask, &v)) continue;
        double den = 1.0;
        if (flat) den *= flat[p];
        if (solidangle) den *= solidangle[p];
        if (polarization) den *= polarization[p];
        double num = image[p] - (dark ? dark[p] : 0.0);
        int n = aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
        if (n > AIO_MAX_SPLIT) return -3;
        for (int k = 0; k < n; ++k) {
            sum_signal[bins[k]] += coefs[k] * num;
            sum_norm[bins[k]] += coefs[k] * den;
        }
    }
    for (int b = 0; b < npt; ++b) intensity[b] = sum_norm[b] != 0.0 ? sum_signal[b] / sum_norm[b] : empty_value;
    return 0;
}

/* O1-O7 from the geometry (single thread). range_or_null = {u0, u1} or NULL for the automatic range. */
int aio_integrate1d(const aio_geometry *g, int height, int width, int npt, int unit, const double *range_or_null,
                    const double *image, const double *dark, const double *flat, const double *solidangle,
                    const double *polarization, const uint8_t *mask, double empty_value,
                    double *radial, double *intensity, double *sum_signal, double *count, double *range_out)
{
    int64_t n = (int64_t)height * width;
    double *u_min = (double *)malloc((size_t)n * sizeof(double));
    double *u_max = (double *)malloc((size_t)n * sizeof(double));
    if (!u_min || !u_max) { free(u_min); free(u_max); return -2; }
    int rc = aio_pixel_bounds(g, height, width, unit, u_min, u_max);
    double u0, u1;
    if (rc == 0) {
        if (range_or_null) { u0 = range_or_null[0]; u1 = range_or_null[1]; }
        else rc = aio_auto_range(u_min, u_max, n, &u0, &u1);
    }
    if (rc == 0) {
        if (range_out) { range_out[0] = u0; range_out[1] = u1; }
        rc = aio_integrate1d_bounds(u_min, u_max, n, npt, u0, u1, image, dark, flat, solidangle, polarization, mask,
                                    empty_value, 1, radial, intensity, sum_signal, count);
    }
    free(u_min); free(u_max);
    return rc;
}

/*
 * The matrix of the "scatter to gather" transformation in scipy-compatible CSR form
 * (data / indices / indptr): the triplets of O4 taken in pixel order and counting-sorted by bin, so
 * that column indices ascend within a row.  Two calls: indices == NULL returns nnz and fills indptr only.
 */
int64_t aio_csr(const double *u_min, const double *u_max, int64_t npix, int npt, double u0, double u1,
                int64_t *indptr, int32_t *indices, double *data)
{
    int bins[AIO_MAX_SPLIT]; double coefs[AIO_MAX_SPLIT];
    int64_t *len = (int64_t *)calloc((size_t)npt + 1, sizeof(int64_t));
    if (!len) return -2;
    for (int64_t p = 0; p < npix; ++p) {
        int n = aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
        if (n > AIO_MAX_SPLIT) { free(len); return -3; }
        for (int k = 0; k < n; ++k) len[bins[k]]++;
    }
    indptr[0] = 0;
    for (int b = 0; b < npt; ++b) indptr[b + 1] = indptr[b] + len[b];
    int64_t nnz = indptr[npt];
    if (indices && data) {
        for (int b = 0; b < npt; ++b) len[b] = indptr[b];      /* running cursors */
        for (int64_t p = 0; p < npix; ++p) {
            int n = aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
            for (int k = 0; k < n; ++k) {
                int64_t pos = len[bins[k]]++;
                indices[pos] = (int32_t)p;
                data[pos] = coefs[k];
            }
        }
    }
    free(len);
    return nnz;
}

/* ==================================================================================================================
 * Bidimensional ("cake") integration: bins = azimuthal x radial ("mono- and bidimensional integration";
 * PAPER.md:114-116, Fig. 3: pixel splitting matters most "when the number of pixels falling into each bin is small like
 * for example for 2D integration").  The paper gives the azimuthal coordinate chi = atan(y/x) and the
 * bounding-box scheme; it says nothing more about the 2D case.  Readings:
 *   - the bounding box is taken in (u, chi): the pixel's extent along each axis, split independently, so that the weight
 *     of pixel p in bin (a, r) is  overlap_chi(a) / w_chi  *  overlap_u(r) / w_u  -- the area of the box segment over
 *     the area of the box ("we use the area of the bounding box segment");
 *   - chi = atan2(y, x) in (-pi, pi]; the azimuthal axis is periodic: a pixel that crosses the negative x axis is
 *     split across the seam, a pixel that holds the beam centre strictly inside covers the full circle;
 *   - default azimuthal range = the full circle [-pi, pi], last bin closed, bins half-open as on the radial axis;
 *   - output layout [npt_azim][npt_rad] (row = azimuthal bin).
 * ================================================================================================================== */

/* Azimuthal extent of pixel (i, j): start chi_lo in [-pi, pi) and width w in [0, 2 pi]; the pixel covers
 * [chi_lo, chi_lo + w], which may run past +pi (the seam).  The extent of a convex region that does not hold the origin
 * is reached at its corners; each corner's angle is measured from the direction of the pixel centre (signed angle
 * atan2(cross, dot)), which keeps the seam out of the way. */
static void pixel_chi_extent(const aio_geometry *g, int i, int j, double *chi_lo, double *chi_w)
{
    const double pi = 3.14159265358979323846;
    double x_lo = ((double)j - g->center_x_px) * g->pixel_x_m;
    double x_hi = ((double)(j + 1) - g->center_x_px) * g->pixel_x_m;
    double y_lo = ((double)i - g->center_y_px) * g->pixel_y_m;
    double y_hi = ((double)(i + 1) - g->center_y_px) * g->pixel_y_m;
    if (x_lo < 0.0 && x_hi > 0.0 && y_lo < 0.0 && y_hi > 0.0) {     /* beam centre strictly inside: every direction */
        *chi_lo = -pi; *chi_w = 2.0 * pi;
        return;
    }
    double xc = 0.5 * (x_lo + x_hi), yc = 0.5 * (y_lo + y_hi);
    double chi_c = atan2(yc, xc);
    double xs[4] = {x_lo, x_hi, x_lo, x_hi}, ys[4] = {y_lo, y_lo, y_hi, y_hi};
    double d_min = 0.0, d_max = 0.0;
    for (int k = 0; k < 4; ++k) {
        if (xs[k] == 0.0 && ys[k] == 0.0) continue;       /* a corner on the beam centre has no direction */
        double d = atan2(xc * ys[k] - yc * xs[k], xc * xs[k] + yc * ys[k]);
        if (d < d_min) d_min = d;
        if (d > d_max) d_max = d;
    }
    double lo = chi_c + d_min;
    if (lo < -pi) lo += 2.0 * pi;
    if (lo >= pi) lo -= 2.0 * pi;
    *chi_lo = lo;
    *chi_w = d_max - d_min;
}

int aio_pixel_chi_bounds(const aio_geometry *g, int height, int width, double *chi_lo, double *chi_w)
{
    if (!g || height < 1 || width < 1) return -1;
    for (int i = 0; i < height; ++i)
        for (int j = 0; j < width; ++j)
            pixel_chi_extent(g, i, j, &chi_lo[(int64_t)i * width + j], &chi_w[(int64_t)i * width + j]);
    return 0;
}

/* Split of the periodic interval [chi_lo, chi_lo + w] over npt bins on [c0, c1] (c1 - c0 <= 2 pi): the interval and its
 * images shifted by -2 pi and +2 pi are each split like a radial interval (aio_split's overlap / width, the width being
 * the pixel's whole w), and what lands in the same bin is added.  Bins come out ascending.  Returns the number of bins. */
int aio_split_azim(double chi_lo, double w, double c0, double c1, int npt, int *bins, double *coefs, int cap)
{
    const double two_pi = 2.0 * 3.14159265358979323846;
    double delta = (c1 - c0) / (double)npt;
    int n = 0;
    if (!(w > 0.0)) {                                   /* degenerate: a direction */
        for (int k = -1; k <= 1; ++k) {
            double f = (chi_lo + two_pi * k - c0) / delta;
            if (f >= 0.0 && f <= (double)npt) {
                int b = (int)floor(f);
                if (b > npt - 1) b = npt - 1;
                if (cap > 0) { bins[0] = b; coefs[0] = 1.0; }
                return 1;
            }
        }
        return 0;
    }
    for (int k = -1; k <= 1; ++k) {
        double f_min = (chi_lo + two_pi * k - c0) / delta;
        double f_max = (chi_lo + w + two_pi * k - c0) / delta;
        double wf = f_max - f_min;                      /* as on the radial axis: width from the two bounds */
        if (!(f_max > 0.0) || !(f_min < (double)npt)) continue;
        double a = max2(f_min, 0.0), z = min2(f_max, (double)npt);
        int b_first = (int)floor(a), b_last = (int)floor(z);
        if (b_last > npt - 1) b_last = npt - 1;
        for (int b = b_first; b <= b_last; ++b) {
            double ov = min2(z, (double)(b + 1)) - max2(a, (double)b);
            if (!(ov > 0.0)) continue;
            int at = -1;
            for (int q = 0; q < n && q < cap; ++q) if (bins[q] == b) at = q;
            if (at >= 0) coefs[at] += ov / wf;
            else {
                if (n < cap) { bins[n] = b; coefs[n] = ov / wf; }
                ++n;
            }
        }
    }
    /* ascending bins (insertion sort: a handful of entries) */
    int m = n < cap ? n : cap;
    for (int q = 1; q < m; ++q) {
        int b = bins[q]; double c = coefs[q]; int t = q - 1;
        while (t >= 0 && bins[t] > b) { bins[t + 1] = bins[t]; coefs[t + 1] = coefs[t]; --t; }
        bins[t + 1] = b; coefs[t + 1] = c;
    }
    return n;
}

/* Forward scatter into azimuthal x radial bins: the 1D loop of aio_integrate1d_bounds with the weight of PAPER.md:120
 * taken on both axes.  Outputs are [npt_azim][npt_rad]. */
int aio_integrate2d_bounds(const double *u_min, const double *u_max, const double *chi_lo, const double *chi_w,
                           int64_t npix, int npt_rad, double u0, double u1, int npt_azim, double c0, double c1,
                           const double *image, const double *dark, const double *flat, const double *solidangle,
                           const double *polarization, const uint8_t *mask, double empty_value,
                           double *intensity, double *sum_signal, double *count)
{
    if (npix < 1 || npt_rad < 1 || npt_azim < 1 || !(u1 > u0) || !(c1 > c0) || !image) return -1;
    int64_t nb = (int64_t)npt_rad * npt_azim;
    int *br = (int *)malloc(AIO_MAX_SPLIT * sizeof(int)), *ba = (int *)malloc(AIO_MAX_SPLIT * sizeof(int));
    double *cr = (double *)malloc(AIO_MAX_SPLIT * sizeof(double)), *ca = (double *)malloc(AIO_MAX_SPLIT * sizeof(double));
    if (!br || !ba || !cr || !ca) { free(br); free(ba); free(cr); free(ca); return -2; }
    for (int64_t b = 0; b < nb; ++b) { sum_signal[b] = 0.0; count[b] = 0.0; }
    int rc = 0;
    for (int64_t p = 0; p < npix && rc == 0; ++p) {
        double v;
        if (!pixel_value(p, image, dark, flat, solidangle, polarization, mask, &v)) continue;
        int nr = aio_split(u_min[p], u_max[p], u0, u1, npt_rad, br, cr, AIO_MAX_SPLIT);
        int na = aio_split_azim(chi_lo[p], chi_w[p], c0, c1, npt_azim, ba, ca, AIO_MAX_SPLIT);
        if (nr > AIO_MAX_SPLIT || na > AIO_MAX_SPLIT) { rc = -3; break; }
        for (int a = 0; a < na; ++a)
            for (int r = 0; r < nr; ++r) {
                int64_t b = (int64_t)ba[a] * npt_rad + br[r];
                sum_signal[b] += ca[a] * cr[r] * v;      /* weighted histogram   */
                count[b] += ca[a] * cr[r];               /* unweighted histogram */
            }
    }
    if (rc == 0)
        for (int64_t b = 0; b < nb; ++b) intensity[b] = count[b] > 0.0 ? sum_signal[b] / count[b] : empty_value;
    free(br); free(ba); free(cr); free(ca);
    return rc;
}

/* The 2D matrix in CSR form: row = a * npt_rad + r, columns (pixels) ascending.  Two calls as aio_csr. */
int64_t aio_csr2d(const double *u_min, const double *u_max, const double *chi_lo, const double *chi_w, int64_t npix,
                  int npt_rad, double u0, double u1, int npt_azim, double c0, double c1,
                  int64_t *indptr, int32_t *indices, double *data)
{
    int64_t nb = (int64_t)npt_rad * npt_azim;
    int *br = (int *)malloc(AIO_MAX_SPLIT * sizeof(int)), *ba = (int *)malloc(AIO_MAX_SPLIT * sizeof(int));
    double *cr = (double *)malloc(AIO_MAX_SPLIT * sizeof(double)), *ca = (double *)malloc(AIO_MAX_SPLIT * sizeof(double));
    int64_t *len = (int64_t *)calloc((size_t)nb + 1, sizeof(int64_t));
    if (!br || !ba || !cr || !ca || !len) { free(br); free(ba); free(cr); free(ca); free(len); return -2; }
    int64_t rc = 0;
    for (int pass = 0; pass < 2 && rc == 0; ++pass) {
        if (pass == 1) {
            indptr[0] = 0;
            for (int64_t b = 0; b < nb; ++b) indptr[b + 1] = indptr[b] + len[b];
            if (!indices || !data) break;
            for (int64_t b = 0; b < nb; ++b) len[b] = indptr[b];      /* running cursors */
        }
        for (int64_t p = 0; p < npix; ++p) {
            int nr = aio_split(u_min[p], u_max[p], u0, u1, npt_rad, br, cr, AIO_MAX_SPLIT);
            int na = aio_split_azim(chi_lo[p], chi_w[p], c0, c1, npt_azim, ba, ca, AIO_MAX_SPLIT);
            if (nr > AIO_MAX_SPLIT || na > AIO_MAX_SPLIT) { rc = -3; break; }
            for (int a = 0; a < na; ++a)
                for (int r = 0; r < nr; ++r) {
                    int64_t b = (int64_t)ba[a] * npt_rad + br[r];
                    if (pass == 0) len[b]++;
                    else {
                        int64_t pos = len[b]++;
                        indices[pos] = (int32_t)p;
                        data[pos] = ca[a] * cr[r];
                    }
                }
        }
    }
    if (rc == 0) rc = indptr[nb];
    free(br); free(ba); free(cr); free(ca); free(len);
    return rc;
}

/* ==================================================================================================================
 * Full pixel splitting (section 4.2): "no abstraction takes place and the pixel splitting works using
 * the area of the actual pixel segments (assuming they are straight lines)".  The pixel is the quadrilateral spanned by
 * its four corners in the (radial unit, chi) plane, sides taken as straight lines; the weight of the pixel in bin b is
 * the area of the part of that quadrilateral between the bin's two edges over the area of the whole quadrilateral.
 * As the paper describes it: "a function for each of the lines that make up the sides of the pixel is defined by
 * calculating the slope and the point of intersection ... the algorithm loops over the bins that the pixel spans over
 * and proceeds to integrate the four functions ... over the bounds of each bin.  Taking the absolute value of the sum of
 * all these integrals will yield the area of the pixel segment".
 * Readings: corner angles are measured from the direction of the pixel centre (no seam); a corner on the beam centre
 * takes the centre direction; a pixel with the beam centre strictly inside, or whose corners are collinear in this plane
 * (zero area), is split by its bounding box instead (section 4.1).
 * ================================================================================================================== */

/* corners (x_lo,y_lo) (x_hi,y_lo) (x_hi,y_hi) (x_lo,y_hi) of pixel (i, j) in the (u, chi) plane; returns 0 if the beam
 * centre is strictly inside the pixel (no quadrilateral) */
static int pixel_corners(const aio_geometry *g, int unit, int i, int j, double u[4], double chi[4])
{
    double x_lo = ((double)j - g->center_x_px) * g->pixel_x_m;
    double x_hi = ((double)(j + 1) - g->center_x_px) * g->pixel_x_m;
    double y_lo = ((double)i - g->center_y_px) * g->pixel_y_m;
    double y_hi = ((double)(i + 1) - g->center_y_px) * g->pixel_y_m;
    if (x_lo < 0.0 && x_hi > 0.0 && y_lo < 0.0 && y_hi > 0.0) return 0;
    double xc = 0.5 * (x_lo + x_hi), yc = 0.5 * (y_lo + y_hi);
    double chi_c = atan2(yc, xc);
    double xs[4] = {x_lo, x_hi, x_hi, x_lo}, ys[4] = {y_lo, y_lo, y_hi, y_hi};
    for (int k = 0; k < 4; ++k) {
        u[k] = unit_of_r(sqrt(xs[k] * xs[k] + ys[k] * ys[k]), g, unit);
        chi[k] = (xs[k] == 0.0 && ys[k] == 0.0) ? chi_c
                                                : chi_c + atan2(xc * ys[k] - yc * xs[k], xc * xs[k] + yc * ys[k]);
    }
    return 1;
}

int aio_pixel_corners(const aio_geometry *g, int height, int width, int unit, double *u4, double *chi4, uint8_t *has_quad)
{
    if (!g || height < 1 || width < 1 || unit < 0 || unit > 4) return -1;
    for (int i = 0; i < height; ++i)
        for (int j = 0; j < width; ++j) {
            int64_t p = (int64_t)i * width + j;
            has_quad[p] = (uint8_t)pixel_corners(g, unit, i, j, u4 + 4 * p, chi4 + 4 * p);
        }
    return 0;
}

/* signed integral of the line through (f_a, c_a) and (f_b, c_b) over the part of [lo, hi] it spans, along its direction */
static double edge_integral(double f_a, double c_a, double f_b, double c_b, double lo, double hi)
{
    if (f_a == f_b) return 0.0;                                  /* a side parallel to the chi axis sweeps no area */
    double m = (c_b - c_a) / (f_b - f_a);                        /* slope; c_a - m f_a is the point of intersection */
    double e_lo = max2(lo, min2(f_a, f_b)), e_hi = min2(hi, max2(f_a, f_b));
    if (!(e_hi > e_lo)) return 0.0;
    double v_lo = c_a + m * (e_lo - f_a), v_hi = c_a + m * (e_hi - f_a);
    double area = 0.5 * (v_lo + v_hi) * (e_hi - e_lo);
    return f_b > f_a ? area : -area;
}

/* full splitting of one quadrilateral; same conventions as aio_split (bins half-open, last closed, returns the count) */
int aio_split_full(const double *u, const double *chi, double u0, double u1, int npt, int *bins, double *coefs, int cap)
{
    double delta = (u1 - u0) / (double)npt, f[4];
    double f_min = 0.0, f_max = 0.0;
    for (int k = 0; k < 4; ++k) {
        f[k] = (u[k] - u0) / delta;
        if (k == 0 || f[k] < f_min) f_min = f[k];
        if (k == 0 || f[k] > f_max) f_max = f[k];
    }
    double total = 0.0;
    for (int k = 0; k < 4; ++k) total += edge_integral(f[k], chi[k], f[(k + 1) & 3], chi[(k + 1) & 3], f_min, f_max);
    total = fabs(total);
    if (!(total > 0.0)) return aio_split(u0 + f_min * delta, u0 + f_max * delta, u0, u1, npt, bins, coefs, cap);
    if (!(f_max > 0.0) || !(f_min < (double)npt)) return 0;
    int b_first = (int)floor(max2(f_min, 0.0)), b_last = (int)floor(min2(f_max, (double)npt)), n = 0;
    if (b_last > npt - 1) b_last = npt - 1;
    for (int b = b_first; b <= b_last; ++b) {
        double area = 0.0;
        for (int k = 0; k < 4; ++k)
            area += edge_integral(f[k], chi[k], f[(k + 1) & 3], chi[(k + 1) & 3], (double)b, (double)(b + 1));
        area = fabs(area);
        if (area > 0.0) {
            if (n < cap) { bins[n] = b; coefs[n] = area / total; }
            ++n;
        }
    }
    return n;
}

/* CSR of the full-splitting matrix (two calls as aio_csr); u_min / u_max are the bounding-box bounds, used for the
 * pixels that have no quadrilateral */
int64_t aio_csr_full(const double *u4, const double *chi4, const uint8_t *has_quad, const double *u_min,
                     const double *u_max, int64_t npix, int npt, double u0, double u1,
                     int64_t *indptr, int32_t *indices, double *data)
{
    int bins[AIO_MAX_SPLIT]; double coefs[AIO_MAX_SPLIT];
    int64_t *len = (int64_t *)calloc((size_t)npt + 1, sizeof(int64_t));
    if (!len) return -2;
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1) {
            indptr[0] = 0;
            for (int b = 0; b < npt; ++b) indptr[b + 1] = indptr[b] + len[b];
            if (!indices || !data) break;
            for (int b = 0; b < npt; ++b) len[b] = indptr[b];
        }
        for (int64_t p = 0; p < npix; ++p) {
            int n = has_quad[p] ? aio_split_full(u4 + 4 * p, chi4 + 4 * p, u0, u1, npt, bins, coefs, AIO_MAX_SPLIT)
                                : aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
            if (n > AIO_MAX_SPLIT) { free(len); return -3; }
            for (int k = 0; k < n; ++k) {
                if (pass == 0) len[bins[k]]++;
                else {
                    int64_t pos = len[bins[k]]++;
                    indices[pos] = (int32_t)p;
                    data[pos] = coefs[k];
                }
            }
        }
    }
    int64_t nnz = indptr[npt];
    free(len);
    return nnz;
}

/*
 * Full pixel splitting, one frame, as the paper states it (section 4.2): a loop over the PIXELS; for each
 * pixel "loops over the bins that the pixel spans", the slice areas give the pixel's contribution to each of those bins
 * (aio_split_full above; the bounding box of aio_split for a pixel without a quadrilateral), and "contributions to the
 * histograms are calculated using these areas": the weighted histogram gets c v, the unweighted one c,
 * v and the pixel's validity from O5 (pixel_value).  Then O7.  A forward scatter like aio_integrate1d_bounds, single
 * thread, plain double sums in pixel order.
 * Pins (tests/test_oracle_pins_full.py): uniform image -> constant profile; sum of sum_signal = sum of v and sum of count
 * = number of valid pixels when the range holds every pixel; npt = 1 -> the mean; masked / invalid pixels
 * leave both histograms; equal to (pinned aio_csr_full matrix) x v; equal to aio_integrate1d_bounds when no pixel has a
 * quadrilateral.
 */
int aio_integrate1d_full(const double *u4, const double *chi4, const uint8_t *has_quad, const double *u_min,
                         const double *u_max, int64_t npix, int npt, double u0, double u1,
                         const double *image, const double *dark, const double *flat, const double *solidangle,
                         const double *polarization, const uint8_t *mask, double empty_value,
                         double *radial, double *intensity, double *sum_signal, double *count)
{
    if (npix < 1 || npt < 1 || !(u1 > u0) || !image) return -1;
    int bins[AIO_MAX_SPLIT]; double coefs[AIO_MAX_SPLIT];
    double delta = (u1 - u0) / (double)npt;
    for (int b = 0; b < npt; ++b) sum_signal[b] = count[b] = 0.0;
    for (int64_t p = 0; p < npix; ++p) {
        double v;
        if (!pixel_value(p, image, dark, flat, solidangle, polarization, mask, &v)) continue;
        int n = has_quad[p] ? aio_split_full(u4 + 4 * p, chi4 + 4 * p, u0, u1, npt, bins, coefs, AIO_MAX_SPLIT)
                            : aio_split(u_min[p], u_max[p], u0, u1, npt, bins, coefs, AIO_MAX_SPLIT);
        if (n > AIO_MAX_SPLIT) return -3;
        for (int k = 0; k < n; ++k) {
            sum_signal[bins[k]] += coefs[k] * v;      /* weighted histogram   */
            count[bins[k]] += coefs[k];               /* unweighted histogram */
        }
    }
    for (int b = 0; b < npt; ++b) {
        if (radial) radial[b] = u0 + ((double)b + 0.5) * delta;
        intensity[b] = count[b] > 0.0 ? sum_signal[b] / count[b] : empty_value;
    }
    return 0;
}

int aio_num_threads_available(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}
