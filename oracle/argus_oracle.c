/*
 * argus_oracle.c -- plain double-precision CPU oracle for the calibrate + HEALPix-resample path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, link or call it.  It shares no code,
 * header, table or helper with paper_2207_14304_b200/ (the CUDA path) and neither imports the other.
 *
 * What it follows.  The paper (PAPER.md, arXiv 2207.14304) states the path in words only:
 *   PAPER.md:141 (sec. 5.1)   "standard image calibrations (dark subtraction, flat fielding, masking of
 *                              bad pixels)" and "a one-directional mapping from celestial to pixel-plane
 *                              coordinates";
 *   PAPER.md:145 (sec. 5.1.1) "Each full-frame image is reprojected into equal-sky-area tiles (based on
 *                              the HEALPix pixelization scheme ...)"; refs [10] PAPER.md:221 (HEALPix) and
 *                              [14] PAPER.md:225 (WCSLIB conventions);
 *   BASELINE.json north_star   the step list (bias, exposure-scaled dark, flat, saturation mask; pix2ang,
 *                              inverse TAN + optional SIP, bilinear / Lanczos-3, value + weight, coadd).
 * The paper prints no formula; each function below restates the standard published definition, written
 * out per output pixel, in angle (trigonometric) form, in the order SURVEY.md section 8(c) O1..O7 lists.
 * The readings taken where the paper is silent are listed in DESIGN.md ("Readings").
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P9 of SURVEY.md 8(c).  Beyond those pins the absolute
 * resampled values are "parity unpinned": the paper gives no worked numeric example.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).  All arithmetic is IEEE
 * double with libm; loops are plain; OpenMP only splits independent output pixels across threads.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288
#define ORC_D2R (ORC_PI / 180.0)

/* wcs array layout (synth.Wcs.as_array): crval[2] deg, crpix[2] px (0-based), cd[4] deg/px row-major,
 * sip_order, ap[36], bp[36] indexed [p*6+q]. */
#define W_CRVAL 0
#define W_CRPIX 2
#define W_CD 4
#define W_ORDER 8
#define W_AP 9
#define W_BP 45

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * O1. Calibration (BASELINE.json north_star: "bias subtraction, exposure-scaled dark
 * subtraction, flat-field division and saturation masking").
 *   cal = (raw - bias - dark * t_exp) / flat
 *   m = 0 if raw >= sat_adu, or bpm != 0, or !(flat >= flat_min) (catches NaN), or any master is
 *   non-finite; else m = 1.  Masked pixels get cal = 0.
 * ------------------------------------------------------------------------------------------------ */
void orc_calibrate(const uint16_t* raw, const float* bias, const float* dark, const float* flat,
                   const uint8_t* bpm, int64_t W, int64_t H, double t_exp, int sat_adu, double flat_min,
                   double* cal, uint8_t* mask) {
    int64_t n = W * H;
    for (int64_t i = 0; i < n; ++i) {
        double r = (double)raw[i], b = (double)bias[i], d = (double)dark[i], f = (double)flat[i];
        int good = 1;
        if ((int)raw[i] >= sat_adu) good = 0;
        if (bpm && bpm[i] != 0) good = 0;
        if (!(f >= flat_min)) good = 0;
        if (!isfinite(b) || !isfinite(d) || !isfinite(f)) good = 0;
        if (good) {
            cal[i] = (r - b - d * t_exp) / f;
            mask[i] = 1;
        } else {
            cal[i] = 0.0;
            mask[i] = 0;
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * O2. Nested index -> (face, ix, iy)  (HEALPix, ref [10] PAPER.md:221).
 *   nside = 2^k, p in [0, 12*4^k): f = p >> 2k; q = p & (4^k - 1); ix = even bits of q, iy = odd bits.
 * ------------------------------------------------------------------------------------------------ */
static int orc_log2(int64_t nside) {
    int k = 0;
    while (((int64_t)1 << k) < nside) ++k;
    return k;
}

void orc_nest2xyf(int64_t nside, int64_t p, int* face, int64_t* ix, int64_t* iy) {
    int k = orc_log2(nside);
    int64_t q = p & ((((int64_t)1) << (2 * k)) - 1);
    int64_t x = 0, y = 0;
    for (int b = 0; b < k; ++b) {
        x |= ((q >> (2 * b)) & 1) << b;
        y |= ((q >> (2 * b + 1)) & 1) << b;
    }
    *face = (int)(p >> (2 * k));
    *ix = x;
    *iy = y;
}

int64_t orc_xyf2nest(int64_t nside, int face, int64_t ix, int64_t iy) {
    int k = orc_log2(nside);
    int64_t q = 0;
    for (int b = 0; b < k; ++b) {
        q |= ((ix >> b) & 1) << (2 * b);
        q |= ((iy >> b) & 1) << (2 * b + 1);
    }
    return ((int64_t)face << (2 * k)) | q;
}

/* ------------------------------------------------------------------------------------------------
 * O3. pix2ang, nested scheme (ref [10]).  Face constants R_f (ring offset) and P_f (phi offset, in
 * units of pi/4).  jr = R_f*nside - ix - iy - 1 is the ring number (1 .. 4 nside - 1).
 *   north cap  (jr <  nside):  nr = jr,           z =  1 - nr^2/(3 nside^2)
 *   belt (nside <= jr <= 3 nside): nr = nside,    z = (2/3)(2 - jr/nside)
 *   south cap  (jr > 3 nside): nr = 4 nside - jr, z = -1 + nr^2/(3 nside^2)
 *   phi = (pi/4) (P_f + (ix - iy)/nr), + 2 pi if negative
 *   sin(theta): caps sqrt(t (2 - t)) with t = nr^2/(3 nside^2) (no cancellation); belt sqrt((1-z)(1+z)).
 *   theta = atan2(sin theta, z).   Sky convention (reading): alpha = phi, delta = pi/2 - theta (ICRS).
 * ------------------------------------------------------------------------------------------------ */
static const int ORC_RF[12] = {2, 2, 2, 2, 3, 3, 3, 3, 4, 4, 4, 4};
static const int ORC_PF[12] = {1, 3, 5, 7, 0, 2, 4, 6, 1, 3, 5, 7};

void orc_pix2ang_nest(int64_t nside, int64_t p, double* theta, double* phi) {
    int face;
    int64_t ix, iy;
    orc_nest2xyf(nside, p, &face, &ix, &iy);
    double ns = (double)nside;
    int64_t jr = (int64_t)ORC_RF[face] * nside - ix - iy - 1;
    double z, sth, nr;
    if (jr < nside) {
        nr = (double)jr;
        double t = nr * nr / (3.0 * ns * ns);
        z = 1.0 - t;
        sth = sqrt(t * (2.0 - t));
    } else if (jr > 3 * nside) {
        nr = (double)(4 * nside - jr);
        double t = nr * nr / (3.0 * ns * ns);
        z = -1.0 + t;
        sth = sqrt(t * (2.0 - t));
    } else {
        nr = ns;
        z = (2.0 / 3.0) * (2.0 - (double)jr / ns);
        sth = sqrt((1.0 - z) * (1.0 + z));
    }
    double ph = (ORC_PI / 4.0) * ((double)ORC_PF[face] + (double)(ix - iy) / nr);
    if (ph < 0.0) ph += 2.0 * ORC_PI;
    *theta = atan2(sth, z);
    *phi = ph;
}

/* ------------------------------------------------------------------------------------------------
 * O3b. ang2pix, nested scheme (ref [10]) -- oracle-only helper used by pins P3..P5.
 * ------------------------------------------------------------------------------------------------ */
static int64_t orc_floor_div(int64_t a, int64_t b) {  /* b > 0 */
    int64_t q = a / b;
    if ((a % b != 0) && (a < 0)) --q;
    return q;
}
static int64_t orc_mod(int64_t a, int64_t b) { return a - orc_floor_div(a, b) * b; }

int64_t orc_ang2pix_nest(int64_t nside, double theta, double phi) {
    double z = cos(theta), za = fabs(z);
    double tt = fmod(phi, 2.0 * ORC_PI);
    if (tt < 0.0) tt += 2.0 * ORC_PI;
    tt = tt / (ORC_PI / 2.0); /* in [0,4) */
    if (tt >= 4.0) tt = 0.0;
    double ns = (double)nside;
    int face;
    int64_t ix, iy;
    if (za <= 2.0 / 3.0) {
        double t1 = ns * (0.5 + tt), t2 = 0.75 * ns * z;
        int64_t jp = (int64_t)floor(t1 - t2), jm = (int64_t)floor(t1 + t2);
        int64_t ifp = orc_floor_div(jp, nside), ifm = orc_floor_div(jm, nside);
        if (ifp == ifm) face = (int)orc_mod(ifp, 4) + 4;
        else if (ifp < ifm) face = (int)orc_mod(ifp, 4);
        else face = (int)orc_mod(ifm, 4) + 8;
        ix = orc_mod(jm, nside);
        iy = nside - 1 - orc_mod(jp, nside);
    } else {
        int64_t ntt = (int64_t)floor(tt);
        if (ntt > 3) ntt = 3;
        double tp = tt - (double)ntt;
        /* sqrt(3 (1 - |z|)) computed from sin^2(theta/2)-style identity to keep precision near poles */
        double sth2 = sin(0.5 * (z > 0 ? theta : ORC_PI - theta));
        double tmp = ns * sqrt(6.0) * sth2; /* 1 - |z| = 2 sin^2(theta'/2) */
        int64_t jp = (int64_t)floor(tp * tmp), jm = (int64_t)floor((1.0 - tp) * tmp);
        if (jp > nside - 1) jp = nside - 1;
        if (jm > nside - 1) jm = nside - 1;
        if (z > 0) {
            face = (int)ntt;
            ix = nside - 1 - jm;
            iy = nside - 1 - jp;
        } else {
            face = (int)ntt + 8;
            ix = jp;
            iy = jm;
        }
    }
    return orc_xyf2nest(nside, face, ix, iy);
}

/* ------------------------------------------------------------------------------------------------
 * O4. Sky -> pixel: inverse gnomonic (TAN) about CRVAL, CD^-1, optional sky->pixel SIP polynomial
 * (AP/BP "inverse" coefficients applied directly; the solver emits a one-directional
 * celestial -> pixel mapping).  WCSLIB conventions (ref [14] PAPER.md:225), LONPOLE = 180 deg.
 *   cos c = sin d0 sin d + cos d0 cos d cos(a - a0)
 *   xi  = cos d sin(a - a0) / cos c                          (radians -> degrees)
 *   eta = (cos d0 sin d - sin d0 cos d cos(a - a0)) / cos c  (radians -> degrees)
 *   (U, V) = CD^-1 (xi, eta)
 *   u = U + sum_{p+q<=order} AP[p][q] U^p V^q,  v = V + sum BP[p][q] U^p V^q   (order > 0)
 *   x = u + crpix0, y = v + crpix1
 * Returns cos c; x, y are only meaningful when cos c > 0.
 * ------------------------------------------------------------------------------------------------ */
double orc_sky2pix(const double* wcs, double alpha, double delta, double* x, double* y) {
    double a0 = wcs[W_CRVAL] * ORC_D2R, d0 = wcs[W_CRVAL + 1] * ORC_D2R;
    double sd0 = sin(d0), cd0 = cos(d0), sd = sin(delta), cdl = cos(delta);
    double da = alpha - a0;
    double cda = cos(da), sda = sin(da);
    double cosc = sd0 * sd + cd0 * cdl * cda;
    if (!(cosc > 0.0)) {
        *x = NAN;
        *y = NAN;
        return cosc;
    }
    double xi = (cdl * sda / cosc) / ORC_D2R;
    double eta = ((cd0 * sd - sd0 * cdl * cda) / cosc) / ORC_D2R;
    double c00 = wcs[W_CD], c01 = wcs[W_CD + 1], c10 = wcs[W_CD + 2], c11 = wcs[W_CD + 3];
    double det = c00 * c11 - c01 * c10;
    double U = (c11 * xi - c01 * eta) / det;
    double V = (-c10 * xi + c00 * eta) / det;
    int order = (int)wcs[W_ORDER];
    double u = U, v = V;
    if (order > 0) {
        double fu = 0.0, fv = 0.0;
        for (int p = 0; p <= order; ++p)
            for (int q = 0; p + q <= order; ++q) {
                double m = pow(U, (double)p) * pow(V, (double)q);
                fu += wcs[W_AP + p * 6 + q] * m;
                fv += wcs[W_BP + p * 6 + q] * m;
            }
        u = U + fu;
        v = V + fv;
    }
    *x = u + wcs[W_CRPIX];
    *y = v + wcs[W_CRPIX + 1];
    return cosc;
}

/* Search-cone radius (reading): rho_max = atan(1.25 * s_rad * hypot(W,H)/2),
 * s = sqrt|det CD| the pixel scale.  Needed so that a polynomial fold-over cannot pull far sky in. */
double orc_cos_rho_max(const double* wcs, int64_t W, int64_t H) {
    double det = wcs[W_CD] * wcs[W_CD + 3] - wcs[W_CD + 1] * wcs[W_CD + 2];
    double s_rad = sqrt(fabs(det)) * ORC_D2R;
    double rho = atan(1.25 * s_rad * hypot((double)W, (double)H) / 2.0);
    return cos(rho);
}

/* nested pixel centre -> frame pixel coordinates (O2+O3+O4).  Returns cos c. */
double orc_pix2xy(const double* wcs, int64_t nside, int64_t p, double* x, double* y) {
    double theta, phi;
    orc_pix2ang_nest(nside, p, &theta, &phi);
    return orc_sky2pix(wcs, phi, ORC_PI / 2.0 - theta, x, y);
}

void orc_pix2xy_many(const double* wcs, int64_t nside, const int64_t* idx, int64_t n, double* x, double* y,
                     double* cosc) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) cosc[i] = orc_pix2xy(wcs, nside, idx[i], &x[i], &y[i]);
}

/* ------------------------------------------------------------------------------------------------
 * O5. Footprint (BASELINE.json north_star: "every HEALPix pixel in the frame footprint").
 * Domain (reading): D = { -0.5 <= x < W - 0.5, -0.5 <= y < H - 0.5 } (the pixel centre falls on the
 * detector; half-open).  F = sorted { p : cos c(p) >= cos rho_max and (x(p), y(p)) in D }.
 * ------------------------------------------------------------------------------------------------ */
static int orc_in_domain(double x, double y, int64_t W, int64_t H) {
    return (x >= -0.5) && (x < (double)W - 0.5) && (y >= -0.5) && (y < (double)H - 0.5);
}

/* exact membership of one pixel + its distance (px) to the domain border (for decision margins) */
int orc_member(const double* wcs, int64_t W, int64_t H, int64_t nside, int64_t p, double cos_rho,
               double* d_border) {
    double x, y;
    double cosc = orc_pix2xy(wcs, nside, p, &x, &y);
    if (!(cosc >= cos_rho)) {
        if (d_border) *d_border = INFINITY;
        return 0;
    }
    int in = orc_in_domain(x, y, W, H);
    if (d_border) {
        double x0 = -0.5, x1 = (double)W - 0.5, y0 = -0.5, y1 = (double)H - 0.5;
        if (in) {
            double d = fmin(fmin(x - x0, x1 - x), fmin(y - y0, y1 - y));
            *d_border = d;
        } else {
            double dx = fmax(fmax(x0 - x, x - x1), 0.0), dy = fmax(fmax(y0 - y, y - y1), 0.0);
            *d_border = hypot(dx, dy);
        }
    }
    return in;
}

/* angular separation (rad) between two sky directions given as (theta, phi); haversine form */
static double orc_angsep(double th1, double ph1, double th2, double ph2) {
    double sdt = sin(0.5 * (th1 - th2)), sdp = sin(0.5 * (ph1 - ph2));
    double h = sdt * sdt + sin(th1) * sin(th2) * sdp * sdp;
    if (h > 1.0) h = 1.0;
    return 2.0 * asin(sqrt(h));
}

/* Recursive descent from the 12 base pixels.  A node at resolution nside_c survives if the angular
 * separation between its centre and CRVAL is <= rho_max + r_pix(nside_c), r_pix = 2/nside_c rad
 * (a deliberately generous bound: the largest centre-to-corner distance of a HEALPix pixel is
 * < 1.1/nside_c).  Every footprint pixel satisfies cos c >= cos rho_max, i.e. lies within rho_max of
 * CRVAL, so no node holding one is ever dropped.  Below split_nside the surviving nodes are expanded
 * exhaustively (every leaf gets the exact predicate).
 *
 * idx_out may be NULL (count only).  Returns the footprint size, or -1 if capacity is too small.
 * min_border receives min over all evaluated leaves of the distance to the domain border (px). */
typedef struct {
    int64_t* v;
    int64_t n, cap;
} orc_vec;
static void orc_push(orc_vec* a, int64_t x) {
    if (a->n == a->cap) {
        a->cap = a->cap ? 2 * a->cap : 1024;
        a->v = (int64_t*)realloc(a->v, (size_t)a->cap * sizeof(int64_t));
    }
    a->v[a->n++] = x;
}

static void orc_descend(const double* wcs, double rho_max, int64_t nside_c, int64_t p, int64_t stop_nside,
                        orc_vec* out) {
    double th, ph;
    orc_pix2ang_nest(nside_c, p, &th, &ph);
    double th0 = ORC_PI / 2.0 - wcs[W_CRVAL + 1] * ORC_D2R, ph0 = wcs[W_CRVAL] * ORC_D2R;
    if (orc_angsep(th, ph, th0, ph0) > rho_max + 2.0 / (double)nside_c) return;
    if (nside_c >= stop_nside) {
        orc_push(out, p);
        return;
    }
    for (int c = 0; c < 4; ++c) orc_descend(wcs, rho_max, 2 * nside_c, 4 * p + c, stop_nside, out);
}

int64_t orc_footprint(const double* wcs, int64_t W, int64_t H, int64_t nside, int64_t split_nside,
                      int64_t* idx_out, int64_t capacity, double* min_border) {
    double cos_rho = orc_cos_rho_max(wcs, W, H);
    double rho_max = acos(cos_rho);
    if (split_nside > nside) split_nside = nside;
    if (split_nside < 1) split_nside = 1;
    orc_vec nodes = {0, 0, 0};
    for (int64_t b = 0; b < 12; ++b) orc_descend(wcs, rho_max, 1, b, split_nside, &nodes); /* ascending */
    int64_t ratio = nside / split_nside, per = ratio * ratio;
    int64_t words = (per + 63) / 64;
    uint64_t* bits = (uint64_t*)calloc((size_t)(nodes.n * words + 1), sizeof(uint64_t));
    int64_t* counts = (int64_t*)calloc((size_t)nodes.n + 1, sizeof(int64_t));
    double dmin = INFINITY;
#pragma omp parallel for schedule(dynamic, 4) reduction(min : dmin)
    for (int64_t i = 0; i < nodes.n; ++i) {
        int64_t base = nodes.v[i] * per, c = 0;
        for (int64_t j = 0; j < per; ++j) {
            double d;
            if (orc_member(wcs, W, H, nside, base + j, cos_rho, &d)) {
                bits[i * words + (j >> 6)] |= ((uint64_t)1) << (j & 63);
                ++c;
            }
            if (d < dmin) dmin = d;
        }
        counts[i] = c;
    }
    int64_t total = 0;
    for (int64_t i = 0; i < nodes.n; ++i) total += counts[i];
    if (min_border) *min_border = dmin;
    if (idx_out) {
        if (total > capacity) {
            total = -1;
        } else {
            int64_t o = 0;
            for (int64_t i = 0; i < nodes.n; ++i) {
                int64_t base = nodes.v[i] * per;
                for (int64_t j = 0; j < per; ++j)
                    if ((bits[i * words + (j >> 6)] >> (j & 63)) & 1) idx_out[o++] = base + j;
            }
        }
    }
    free(bits);
    free(counts);
    free(nodes.v);
    return total;
}

/* ------------------------------------------------------------------------------------------------
 * O6. Interpolation (BASELINE.json north_star: "bilinear or Lanczos-3 interpolation, and write a
 * per-pixel value and weight").  i0 = floor(x), fx = x - i0 (same in y).
 *   bilinear : columns i0, i0+1, kx = (1 - fx, fx)
 *   Lanczos-3: columns i0-2 .. i0+3, kx_i = L(x - i), L(t) = sinc(t) sinc(t/3) for |t| < 3 else 0,
 *              sinc(t) = sin(pi t)/(pi t), L(0) = 1
 *   2-D tap weight k = kx * ky.  Taps outside the frame count as m = 0.
 *   S0 = sum k (all taps), B = sum k (1 - m), V1 = sum k m cal, w = 1 - B/S0
 *   if w < w_min: (value, weight) = (0, 0) else value = V1/(S0 - B), weight = min(w, 1).
 * (Reading: weight = fraction of kernel mass on good in-frame pixels; value renormalised by the good
 * kernel mass.)  *flag gets bit 0 = "margin-ambiguous" (x or y within 1e-4 px of an integer AND a bad
 * tap in either adjacent cell's tap set; or |w - w_min| < 1e-4): such pixels are excluded from value
 * parity (the interpolant is discontinuous there).
 * ------------------------------------------------------------------------------------------------ */
#define ORC_BILINEAR 0
#define ORC_LANCZOS3 1

static double orc_sinc(double t) {
    if (t == 0.0) return 1.0;
    double a = ORC_PI * t;
    return sin(a) / a;
}
static double orc_lanczos3(double t) {
    if (fabs(t) >= 3.0) return 0.0;
    return orc_sinc(t) * orc_sinc(t / 3.0);
}

static int orc_tap_good(const uint8_t* mask, int64_t W, int64_t H, int64_t i, int64_t j) {
    if (i < 0 || i >= W || j < 0 || j >= H) return 0;
    return mask[j * W + i] != 0;
}

/* any bad tap in the tap set anchored at cell (i0, j0)? */
static int orc_any_bad(const uint8_t* mask, int64_t W, int64_t H, int64_t i0, int64_t j0, int lo, int hi) {
    for (int dj = lo; dj <= hi; ++dj)
        for (int di = lo; di <= hi; ++di)
            if (!orc_tap_good(mask, W, H, i0 + di, j0 + dj)) return 1;
    return 0;
}

void orc_interp(const double* cal, const uint8_t* mask, int64_t W, int64_t H, double x, double y, int kernel,
                double w_min, double* value, double* weight, uint8_t* flag) {
    int lo = (kernel == ORC_LANCZOS3) ? -2 : 0, hi = (kernel == ORC_LANCZOS3) ? 3 : 1;
    double fi = floor(x), fj = floor(y);
    int64_t i0 = (int64_t)fi, j0 = (int64_t)fj;
    double fx = x - fi, fy = y - fj;
    double kx[6], ky[6];
    int nt = hi - lo + 1;
    if (kernel == ORC_LANCZOS3) {
        for (int t = 0; t < nt; ++t) {
            kx[t] = orc_lanczos3(x - (double)(i0 + lo + t));
            ky[t] = orc_lanczos3(y - (double)(j0 + lo + t));
        }
    } else {
        kx[0] = 1.0 - fx;
        kx[1] = fx;
        ky[0] = 1.0 - fy;
        ky[1] = fy;
    }
    double S0 = 0.0, B = 0.0, V1 = 0.0;
    for (int tj = 0; tj < nt; ++tj)
        for (int ti = 0; ti < nt; ++ti) {
            double k = kx[ti] * ky[tj];
            int64_t i = i0 + lo + ti, j = j0 + lo + tj;
            S0 += k;
            if (orc_tap_good(mask, W, H, i, j)) V1 += k * cal[j * W + i];
            else B += k;
        }
    double w = 1.0 - B / S0;
    if (w < w_min) {
        *value = 0.0;
        *weight = 0.0;
    } else {
        *value = V1 / (S0 - B);
        *weight = (w < 1.0) ? w : 1.0;
    }
    if (flag) {
        uint8_t f = 0;
        double eps = 1e-4;
        int near_x = (fx < eps) || (fx > 1.0 - eps), near_y = (fy < eps) || (fy > 1.0 - eps);
        if (near_x || near_y) {
            /* the neighbouring cells whose tap sets the point could fall into */
            for (int dj = -1; dj <= 1 && !f; ++dj)
                for (int di = -1; di <= 1 && !f; ++di) {
                    if (di && !near_x) continue;
                    if (dj && !near_y) continue;
                    if (di == -1 && !(fx < eps)) continue;
                    if (di == 1 && !(fx > 1.0 - eps)) continue;
                    if (dj == -1 && !(fy < eps)) continue;
                    if (dj == 1 && !(fy > 1.0 - eps)) continue;
                    if (orc_any_bad(mask, W, H, i0 + di, j0 + dj, lo, hi)) f = 1;
                }
        }
        /* B == 0 gives w == 1 exactly on any implementation: not ambiguous even when w_min == 1 */
        if (B != 0.0 && fabs(w - w_min) < eps) f = 1;
        *flag = f;
    }
}

/* ------------------------------------------------------------------------------------------------
 * Whole path per output pixel (O2..O6), on an already calibrated frame (O1 output).
 * idx: nested indices (any order); outputs value[n], weight[n] (double), flag[n] (may be NULL),
 * xs/ys (may be NULL) the source coordinates.
 * ------------------------------------------------------------------------------------------------ */
void orc_resample(const double* cal, const uint8_t* mask, int64_t W, int64_t H, const double* wcs,
                  int64_t nside, int kernel, double w_min, const int64_t* idx, int64_t n, double* value,
                  double* weight, uint8_t* flag, double* xs, double* ys) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double x, y;
        double cosc = orc_pix2xy(wcs, nside, idx[i], &x, &y);
        if (xs) xs[i] = x;
        if (ys) ys[i] = y;
        if (!(cosc > 0.0) || !isfinite(x) || !isfinite(y) || fabs(x) > 1e9 || fabs(y) > 1e9) {
            value[i] = 0.0;
            weight[i] = 0.0;
            if (flag) flag[i] = 0;
            continue;
        }
        orc_interp(cal, mask, W, H, x, y, kernel, w_min, &value[i], &weight[i], flag ? &flag[i] : NULL);
    }
}

/* ------------------------------------------------------------------------------------------------
 * O7. Coadd accumulate (BASELINE.json configs[3]: "sum/weight-accumulated into a single HEALPix coadd
 * buffer"; tiles are pre-aligned to a fixed HEALPix grid).
 * Layout: sorted tile ids at resolution nside_tile (NSIDE = 256 in PAPER.md:145); each tile holds
 * ppt = (nside/nside_tile)^2 consecutive nested pixels: slot(p) = rank(p / ppt) * ppt + (p mod ppt).
 *   sum[slot] += w * v;  wsum[slot] += w.   Pixels whose tile is absent are skipped and counted.
 * ------------------------------------------------------------------------------------------------ */
int64_t orc_coadd_accumulate(const int64_t* tiles, int64_t n_tiles, int64_t ppt, double* sum, double* wsum,
                             const int64_t* idx, const double* value, const double* weight, int64_t n) {
    int64_t skipped = 0;
    for (int64_t i = 0; i < n; ++i) {
        int64_t t = idx[i] / ppt, r = idx[i] % ppt;
        int64_t lo = 0, hi = n_tiles - 1, pos = -1;
        while (lo <= hi) {
            int64_t mid = (lo + hi) / 2;
            if (tiles[mid] == t) { pos = mid; break; }
            if (tiles[mid] < t) lo = mid + 1; else hi = mid - 1;
        }
        if (pos < 0) { ++skipped; continue; }
        sum[pos * ppt + r] += weight[i] * value[i];
        wsum[pos * ppt + r] += weight[i];
    }
    return skipped;
}
