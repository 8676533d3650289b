/*
 * dt_oracle.c -- CPU ORACLE (test infrastructure; see dt_oracle.h for scope, pins and rules).
 *
 * Plain C, IEEE fp64, build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared.
 * Each function cites the step of SURVEY.md section 8(c) ("the definition") it evaluates; those
 * steps restate BASELINE.json north_star, the paper giving only the skeleton (PAPER.md:141-143,
 * PAPER.md:202, Algorithm 1).
 */
#include "dt_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double DTO_PI = 3.14159265358979323846;
static const double DTO_TWO_PI = 6.28318530717958647692;

int dto_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int valid_orbit(const double el[6])
{
    for (int k = 0; k < 6; ++k)
        if (!isfinite(el[k])) return 0;
    return el[0] > 0.0 && el[1] >= 0.0 && el[1] < 1.0;
}

/* Step 2 (8(c).2, readings A4/A5): m = M - 2pi*round(M/2pi); fold to [0, pi]; E0 = min(m + e, pi)
 * (f convex on [0, pi] and f(E0) >= 0, so Newton descends monotonically);
 * E <- E - (E - e sinE - m)/(1 - e cosE) until |dE| <= 1e-15 max(1,|E|) or 50 iterations. */
int dto_kepler(double e, double M, double *E_out, int32_t *iters, double *resid)
{
    if (!(e >= 0.0 && e < 1.0) || !isfinite(M)) return -1;
    double m = M - DTO_TWO_PI * round(M / DTO_TWO_PI);
    double sigma = (m < 0.0) ? -1.0 : 1.0;
    m = fabs(m);
    double E = fmin(m + e, DTO_PI);
    int it = 0;
    for (it = 1; it <= 50; ++it) {
        double dE = (E - e * sin(E) - m) / (1.0 - e * cos(E));
        E = E - dE;
        if (fabs(dE) <= 1e-15 * fmax(1.0, fabs(E))) break;
    }
    if (iters) *iters = it > 50 ? 50 : it;
    if (resid) *resid = fabs(E - e * sin(E) - m);
    *E_out = sigma * E;
    return 0;
}

/* Step 3 basis (8(c).3): perifocal unit vectors in the heliocentric ecliptic frame. */
void dto_pq(double inc, double node, double peri, double P[3], double Q[3])
{
    double ci = cos(inc), si = sin(inc);
    double cO = cos(node), sO = sin(node);
    double cw = cos(peri), sw = sin(peri);
    P[0] = cO * cw - sO * sw * ci;
    P[1] = sO * cw + cO * sw * ci;
    P[2] = sw * si;
    Q[0] = -cO * sw - sO * cw * ci;
    Q[1] = -sO * sw + cO * cw * ci;
    Q[2] = cw * si;
}

/* Steps 1-3 (8(c).1-3): n = sqrt(GM/a^3); M = M0 + n (t - t0); solve Kepler;
 * r = a (cosE - e) P + a sqrt(1 - e^2) sinE Q. */
static int helio_full(const double el[6], double gm, double t, double t0, double r[3],
                      double *M_out, double *E_out, int32_t *iters, double *resid)
{
    double a = el[0], e = el[1];
    double n = sqrt(gm / (a * a * a));
    double M = el[5] + n * (t - t0);
    double E;
    if (dto_kepler(e, M, &E, iters, resid) != 0) return -1;
    double P[3], Q[3];
    dto_pq(el[2], el[3], el[4], P, Q);
    double X = a * (cos(E) - e);
    double Y = a * sqrt(1.0 - e * e) * sin(E);
    for (int k = 0; k < 3; ++k) r[k] = X * P[k] + Y * Q[k];
    if (M_out) *M_out = M;
    if (E_out) *E_out = E;
    return 0;
}

int dto_helio(const double el[6], double gm, double t, double t0, double r[3], double *M_out,
              double *E_out)
{
    return helio_full(el, gm, t, t0, r, M_out, E_out, NULL, NULL);
}

static void nan_pair(dto_pair *o)
{
    memset(o, 0, sizeof *o);
    double q = NAN;
    o->M = o->E = o->tau = o->M1 = o->E1 = o->rho = o->ra = o->dec = q;
    o->D = o->xi = o->eta = o->x = o->y = q;
    for (int k = 0; k < 3; ++k) o->r[k] = o->r1[k] = o->q[k] = q;
    o->ix = o->iy = -1;
}

/* Steps 1-8 for one pair (8(c).1-8; readings A6-A11). */
int dto_pair_chain(const dto_survey *s, const double el[6], double t0, int32_t j, dto_pair *o)
{
    if (!valid_orbit(el)) { nan_pair(o); return -1; }
    memset(o, 0, sizeof *o);
    const double t = s->t[j];
    const double *R = s->obs_ecl + 3 * (int64_t)j;
    /* steps 1-3 at time t */
    double res0 = 0.0, res1 = 0.0;
    helio_full(el, s->gm, t, t0, o->r, &o->M, &o->E, &o->kepler_iters, &res0);

    /* step 4 (A6): exactly one light-time iteration; the observer stays at t */
    double d0[3];
    for (int k = 0; k < 3; ++k) d0[k] = o->r[k] - R[k];
    o->tau = sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2]) / s->c;
    helio_full(el, s->gm, t - o->tau, t0, o->r1, &o->M1, &o->E1, NULL, &res1);
    o->kepler_resid = res0 > res1 ? res0 : res1;

    /* step 5 (A7, A8): topocentric, then ecliptic -> equatorial */
    double d[3];
    for (int k = 0; k < 3; ++k) d[k] = o->r1[k] - R[k];
    double ce = cos(s->obliquity), se = sin(s->obliquity);
    o->q[0] = d[0];
    o->q[1] = d[1] * ce - d[2] * se;
    o->q[2] = d[1] * se + d[2] * ce;

    /* step 6: sky position */
    o->rho = sqrt(o->q[0] * o->q[0] + o->q[1] * o->q[1] + o->q[2] * o->q[2]);
    o->ra = atan2(o->q[1], o->q[0]);
    if (o->ra < 0.0) o->ra += DTO_TWO_PI;
    o->dec = asin(o->q[2] / o->rho);

    /* step 7 (A9, A10): gnomonic projection, textbook trigonometric form */
    double a0 = s->ra0[j], d0t = s->dec0[j];
    double sd0 = sin(d0t), cd0 = cos(d0t), sd = sin(o->dec), cd = cos(o->dec);
    double cda = cos(o->ra - a0), sda = sin(o->ra - a0);
    o->D = sd0 * sd + cd0 * cd * cda;
    o->xi = cd * sda / o->D;
    o->eta = (cd0 * sd - sd0 * cd * cda) / o->D;

    /* step 8 (A9, A11): pixel coordinates, footprint test in floating point, nearest pixel */
    double W = (double)s->width, H = (double)s->height;
    o->x = (W - 1.0) / 2.0 + o->xi / s->pixel_scale;
    o->y = (H - 1.0) / 2.0 + o->eta / s->pixel_scale;
    double xh = o->x + 0.5, yh = o->y + 0.5;
    o->hit = (o->D > 0.0 && xh >= 0.0 && xh < W && yh >= 0.0 && yh < H) ? 1 : 0;
    if (o->hit) {
        o->ix = (int32_t)floor(xh);
        o->iy = (int32_t)floor(yh);
    } else {
        o->ix = o->iy = -1;
    }
    o->flag = 0;
    if (o->D > 0.0 && isfinite(xh) && isfinite(yh) && fabs(xh) < 1e15 && fabs(yh) < 1e15) {
        double fx = xh - floor(xh), fy = yh - floor(yh);
        if (fx < 1e-6 || fx > 1.0 - 1e-6 || fy < 1e-6 || fy > 1.0 - 1e-6) o->flag = 1;
    }
    return 0;
}

int dto_project(const dto_survey *s, const double *elements, int64_t n, double t0,
                double *radec, double *xy, int32_t *pix, uint8_t *flag)
{
    const int32_t N = s->n_exposures;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t o = 0; o < n; ++o) {
        for (int32_t j = 0; j < N; ++j) {
            dto_pair p;
            dto_pair_chain(s, elements + 6 * o, t0, j, &p);
            int64_t k = o * N + j;
            if (radec) { radec[2 * k] = p.ra; radec[2 * k + 1] = p.dec; }
            if (xy) { xy[2 * k] = p.x; xy[2 * k + 1] = p.y; }
            if (pix) { pix[2 * k] = p.ix; pix[2 * k + 1] = p.iy; }
            if (flag) flag[k] = (uint8_t)p.flag;
        }
    }
    return 0;
}

/* Steps 9-10 (8(c).9-10; A12-A17): in ascending exposure index
 * S += f / v; Wt += 1 / v; n_hit += 1 (masked pixels skipped); SNR = S / sqrt(Wt), 0 if no hit. */
int dto_stack(const dto_survey *s, const float *const *flux, const float *const *var,
              const double *elements, int64_t n, double t0,
              double *snr, int32_t *hits, double *S_out, double *Wt_out, int32_t *nflag)
{
    const int32_t N = s->n_exposures;
    const int64_t W = s->width;
    if (s->variance_mode == 1 && var == NULL) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t o = 0; o < n; ++o) {
        const double *el = elements + 6 * o;
        if (!valid_orbit(el)) {
            if (snr) snr[o] = NAN;
            if (hits) hits[o] = -1;
            if (S_out) S_out[o] = NAN;
            if (Wt_out) Wt_out[o] = NAN;
            if (nflag) nflag[o] = 0;
            continue;
        }
        double S = 0.0, Wt = 0.0;
        int32_t nh = 0, nf = 0;
        for (int32_t j = 0; j < N; ++j) {
            dto_pair p;
            dto_pair_chain(s, el, t0, j, &p);
            if (p.flag && p.D > 0.0 && p.x + 0.5 >= -1.0 && p.x + 0.5 < (double)s->width + 1.0 &&
                p.y + 0.5 >= -1.0 && p.y + 0.5 < (double)s->height + 1.0)
                nf += 1;
            if (!p.hit) continue;
            int64_t off = (int64_t)p.iy * W + p.ix;
            double f = (double)flux[j][off];
            double v = (s->variance_mode == 1) ? (double)var[j][off] : s->var_scalar[j];
            if (!(isfinite(f) && isfinite(v) && v > 0.0)) continue;
            S += f / v;
            Wt += 1.0 / v;
            nh += 1;
        }
        if (snr) snr[o] = (nh > 0) ? S / sqrt(Wt) : 0.0;
        if (hits) hits[o] = nh;
        if (S_out) S_out[o] = S;
        if (Wt_out) Wt_out[o] = Wt;
        if (nflag) nflag[o] = nf;
    }
    return 0;
}

/* SURVEY.md 8(f) NEXT-1 / NEXT-3 (readings A21-A23): patch gather with PSF weights, per-intersection
 * outlier rejection, per-orbit epochs.  See dt_oracle.h for the definition this follows line by line. */
int dto_stack_ex(const dto_survey *s, const float *const *flux, const float *const *var,
                 const double *elements, int64_t n, double t0, const dto_stack_opts *opts,
                 double *snr, int32_t *hits, double *S_out, double *Wt_out, int32_t *nflag)
{
    const int32_t N = s->n_exposures;
    const int64_t W = s->width, H = s->height;
    const int32_t k = opts ? opts->patch : 1;
    if (k < 1 || (k % 2) == 0) return -1;
    if (s->variance_mode == 1 && var == NULL) return -1;
    const int32_t h = k / 2;
    const double clip = opts ? opts->clip : INFINITY;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t o = 0; o < n; ++o) {
        const double *el = elements + 6 * o;
        const double t0o = (opts && opts->t0_per_orbit) ? opts->t0_per_orbit[o] : t0;
        if (!valid_orbit(el) || !isfinite(t0o)) {
            if (snr) snr[o] = NAN;
            if (hits) hits[o] = -1;
            if (S_out) S_out[o] = NAN;
            if (Wt_out) Wt_out[o] = NAN;
            if (nflag) nflag[o] = 0;
            continue;
        }
        double S = 0.0, Wt = 0.0;
        int32_t nh = 0, nf = 0;
        for (int32_t j = 0; j < N; ++j) {
            dto_pair p;
            dto_pair_chain(s, el, t0o, j, &p);
            if (p.flag && p.D > 0.0 && p.x + 0.5 >= -1.0 && p.x + 0.5 < (double)s->width + 1.0 &&
                p.y + 0.5 >= -1.0 && p.y + 0.5 < (double)s->height + 1.0)
                nf += 1;
            if (!p.hit) continue;
            double si = 0.0, wti = 0.0;
            int32_t used = 0;
            for (int32_t dy = -h; dy <= h; ++dy) {
                for (int32_t dx = -h; dx <= h; ++dx) {
                    const int64_t yy = (int64_t)p.iy + dy, xx = (int64_t)p.ix + dx;
                    if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                    const int64_t off = yy * W + xx;
                    const double f = (double)flux[j][off];
                    const double v = (s->variance_mode == 1) ? (double)var[j][off] : s->var_scalar[j];
                    if (!(isfinite(f) && isfinite(v) && v > 0.0)) continue;
                    const double w = (opts && opts->weights) ? opts->weights[(dy + h) * k + (dx + h)] : 1.0;
                    si += (w * f) / v;
                    wti += (w * w) / v;
                    used += 1;
                }
            }
            if (used == 0) continue;
            if (si > clip * sqrt(wti)) continue;
            S += si;
            Wt += wti;
            nh += 1;
        }
        if (snr) snr[o] = (nh > 0) ? S / sqrt(Wt) : 0.0;
        if (hits) hits[o] = nh;
        if (S_out) S_out[o] = S;
        if (Wt_out) Wt_out[o] = Wt;
        if (nflag) nflag[o] = nf;
    }
    return 0;
}

/* Threshold mode (reading A24): plain scan in ascending orbit index. */
int dto_threshold(const double *snr, const int32_t *hits, int64_t n, double snr_min, int32_t min_hits,
                  int64_t max_out, int64_t *index_out, double *snr_out, int64_t *n_found)
{
    if (max_out < 0 || !n_found) return -1;
    int64_t m = 0;
    for (int64_t o = 0; o < n; ++o) {
        if (!(isfinite(snr[o]) && snr[o] >= snr_min && hits[o] >= min_hits)) continue;
        if (m < max_out) {
            if (index_out) index_out[m] = o;
            if (snr_out) snr_out[m] = snr[o];
        }
        ++m;
    }
    *n_found = m;
    return 0;
}

/* Step 11 (8(c).11): full sort, SNR descending, ties by orbit index ascending. */
typedef struct { double snr; int64_t idx; } dto_cand;

static int cand_cmp(const void *pa, const void *pb)
{
    const dto_cand *a = (const dto_cand *)pa, *b = (const dto_cand *)pb;
    if (a->snr > b->snr) return -1;
    if (a->snr < b->snr) return 1;
    return (a->idx > b->idx) - (a->idx < b->idx);
}

int dto_topk(const double *snr, const int32_t *hits, int64_t n, int32_t k, int32_t min_hits,
             int64_t *index_out, double *snr_out, int32_t *n_found)
{
    if (k < 0) return -1;
    dto_cand *c = (dto_cand *)malloc((size_t)(n > 0 ? n : 1) * sizeof *c);
    if (!c) return -2;
    int64_t m = 0;
    for (int64_t o = 0; o < n; ++o)
        if (hits[o] >= min_hits && isfinite(snr[o])) { c[m].snr = snr[o]; c[m].idx = o; ++m; }
    qsort(c, (size_t)m, sizeof *c, cand_cmp);
    int32_t out = (int32_t)((m < (int64_t)k) ? m : (int64_t)k);
    for (int32_t r = 0; r < out; ++r) { index_out[r] = c[r].idx; snr_out[r] = c[r].snr; }
    *n_found = out;
    free(c);
    return 0;
}
