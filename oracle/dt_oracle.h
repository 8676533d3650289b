/*
 * dt_oracle.h -- CPU ORACLE for the non-linear digital-tracking hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA library under paper_2503_08854_b200/csrc (and neither
 * includes the other).
 *
 * What it is: the plain definition of what the path computes, evaluated pair by pair in IEEE fp64
 * (compile with -O2 -ffp-contract=off, no -ffast-math), in the order and notation of
 * SURVEY.md section 8(c) steps 1-11, which restate BASELINE.json `north_star` (the paper prints no
 * formula for any step: PAPER.md:141-143 and PAPER.md:202 give only the skeleton "orbital
 * parameters -> sky position at the image time -> location in the pixel grid -> keep in-image
 * intersections -> pull pixels -> combine per-orbit signal", Algorithm 1).
 * The only parallelism is an OpenMP `parallel for` over orbits; nothing is blocked, fused or
 * reordered.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 Kepler residual, P2 Kepler values,
 * P3 circular closed form, P4 invariants, P5 light-time closed form, P6 frame + sky closed form,
 * P7 gnomonic identities, P8 worked example WE-1, P9 stack identities / brute force / injected
 * source recovery, P10 top-k vs full sort, A11 guard-band flag and nflag, P11 extended stack (patch,
 * outlier clip, per-orbit epochs) and threshold mode (tests/test_oracle_next.py).  Parity unpinned: anything about real ZTF pixels,
 * Chiron's recovered SNR, the Fig. 3 histogram (data and the paper's Python pipeline are missing).
 *
 * Units: AU, days, radians.
 */
#ifndef DT_ORACLE_H
#define DT_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t n_exposures, width, height;
    const double *t;        /* [N] exposure mid-times, days */
    const double *obs_ecl;  /* [N][3] heliocentric ecliptic observer position, AU */
    const double *ra0;      /* [N] tangent point right ascension, rad */
    const double *dec0;     /* [N] tangent point declination, rad */
    double pixel_scale;     /* rad / pixel */
    double gm;              /* AU^3 / day^2 */
    double c;               /* AU / day; +inf => no light-time */
    double obliquity;       /* rad */
    int32_t variance_mode;  /* 0: per-exposure scalar; 1: fp32 plane per exposure */
    const double *var_scalar; /* [N], mode 0 */
} dto_survey;

/* every intermediate of the chain for one (orbit, exposure) pair: steps 1-8 */
typedef struct {
    double M, E;            /* step 1-2 at time t */
    double r[3];            /* step 3: heliocentric ecliptic position at t */
    double tau;             /* step 4: light-time, days */
    double M1, E1;          /* step 4: mean / eccentric anomaly at t - tau */
    double r1[3];           /* step 4: heliocentric ecliptic position at t - tau */
    double q[3];            /* step 5: topocentric equatorial vector */
    double rho, ra, dec;    /* step 6 */
    double D, xi, eta;      /* step 7 */
    double x, y;            /* step 8: 0-based pixel-centre coordinates */
    int32_t ix, iy;         /* nearest pixel, (-1,-1) when culled */
    int32_t hit;            /* 1 iff inside the footprint and D > 0 */
    int32_t flag;           /* 1 iff x+1/2 or y+1/2 lies within 1e-6 of an integer (A11) */
    int32_t kepler_iters;   /* Newton iterations of the first solve */
    double kepler_resid;    /* max |E - e sinE - m| over both solves (P1) */
} dto_pair;

/* step 2: solve E - e sin E = M. Returns 0, or -1 if e is outside [0,1) or input non-finite. */
int dto_kepler(double e, double M, double *E, int32_t *iters, double *resid);

/* step 3 basis: P, Q from (i, Omega, omega) */
void dto_pq(double inc, double node, double peri, double P[3], double Q[3]);

/* steps 1-3: heliocentric ecliptic position at time t */
int dto_helio(const double el[6], double gm, double t, double t0, double r[3], double *M, double *E);

/* steps 1-8 for one pair */
int dto_pair_chain(const dto_survey *s, const double el[6], double t0, int32_t j, dto_pair *out);

/* steps 1-8 for all pairs.  Any output pointer may be NULL.
 * radec [n][N][2], xy [n][N][2], pix [n][N][2] ((-1,-1) when culled), flag [n][N] (uint8). */
int dto_project(const dto_survey *s, const double *elements, int64_t n, double t0,
                double *radec, double *xy, int32_t *pix, uint8_t *flag);

/* steps 1-10.  flux[j], var[j] point to [H][W] fp32 planes (var may be NULL in mode 0).
 * Outputs (any may be NULL): snr[n], hits[n], S[n], Wt[n], nflag[n] (flagged hits or near-hits). */
int dto_stack(const dto_survey *s, const float *const *flux, const float *const *var,
              const double *elements, int64_t n, double t0,
              double *snr, int32_t *hits, double *S, double *Wt, int32_t *nflag);

/* ---- SURVEY.md 8(f) NEXT rows (readings A21-A24 of DESIGN.md; the paper gives prose only) -------------
 * Options of the extended stack.  For every intersection i (a pair that passes the footprint test of
 * step 8, nearest pixel (ix, iy)) the k x k patch of pixels centred on (ix, iy) is read ("a
 * patch of pixels is pulled from the associated image"), row by row (dy ascending, then dx ascending):
 *     for each patch pixel p inside the image with finite f_p, v_p and v_p > 0:
 *         s_i += (w_p * f_p) / v_p;   wt_i += (w_p * w_p) / v_p;          (s_i, wt_i start at 0)
 * (matched filter with caller-supplied PSF weights w[k*k], row-major; v_p is the exposure's scalar in
 * variance mode 0).  The intersection is skipped (not counted) when no patch pixel contributed, or when
 * its own SNR is anomalously high ("Intersections with anomalously high SNR value compared
 * to the expectation can be removed"):  s_i > clip * sqrt(wt_i)  (clip = +inf: never).  Otherwise, in
 * ascending exposure order, S += s_i; Wt += wt_i; hits += 1.  SNR = S / sqrt(Wt), 0 without hits.
 * patch = 1, weights = {1}, clip = +inf, t0_per_orbit = NULL is dto_stack bit for bit.
 * t0_per_orbit ("six orbital elements and an orbital epoch"): epoch of orbit o's M0, or NULL
 * for the scalar t0 argument. */
typedef struct {
    int32_t patch;                /* k >= 1, odd */
    const double *weights;        /* [k*k] row-major (dy, dx); NULL => all 1 */
    double clip;                  /* +inf => no rejection */
    const double *t0_per_orbit;   /* [n] or NULL */
} dto_stack_opts;

int dto_stack_ex(const dto_survey *s, const float *const *flux, const float *const *var,
                 const double *elements, int64_t n, double t0, const dto_stack_opts *opts,
                 double *snr, int32_t *hits, double *S, double *Wt, int32_t *nflag);

/* Threshold mode of `FindSignificantResults` (Alg. 1; "detections above an SNR of 5",
 * PAPER.md:336): every orbit with finite snr >= snr_min and hits >= min_hits, in ascending orbit index.
 * *n_found = how many there are; the first min(*n_found, max_out) are written. */
int dto_threshold(const double *snr, const int32_t *hits, int64_t n, double snr_min, int32_t min_hits,
                  int64_t max_out, int64_t *index_out, double *snr_out, int64_t *n_found);

/* step 11: k largest SNR among orbits with hits >= min_hits and finite SNR; ties by index. */
int dto_topk(const double *snr, const int32_t *hits, int64_t n, int32_t k, int32_t min_hits,
             int64_t *index_out, double *snr_out, int32_t *n_found);

int dto_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
