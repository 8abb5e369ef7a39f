/*
 * sht_oracle.c -- CPU ORACLE for the batched HEALPix spherical-harmonic transforms of
 * arXiv:2208.10154 ("Accelerating spherical harmonic transforms for a large number of sky maps").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA library (paper_2208_10154_b200/csrc, include/sht.h).
 *
 * It is the *plain definition* of the transforms, written out: per-pixel DFT phases (no FFT, no
 * frequency-circle aliasing rule, no bins), its own normalised Legendre recurrence carried with an
 * explicit extended exponent (no dependence on any underflow trick), no north/south folding, no ring
 * pruning, long double accumulation.  Every function cites the passage of PAPER.md it follows; where
 * the paper defers to HEALPix the reading is the one listed in DESIGN.md
 * ("Readings of the paper") and pinned in tests/ by closed forms, scipy's sph_harm_y and brute force.
 *
 * Layouts (identical to the C ABI so the same seeded arrays feed both sides):
 *   maps : [nmaps][ncomp][npix]      double, HEALPix RING order, ncomp = 1 (T) or 2 (Q,U)
 *   alm  : [nmaps][ncomp][nalm][2]   double (re,im), m >= 0 only, m-major:
 *          idx(l,m) = m(2 lmax + 1 - m)/2 + l, ncomp order (E,B) for spin 2.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_*.py, except the absolute values of
 * the per-iteration residual rms of oracle_analysis_iter, which the paper does not print
 * ("parity unpinned": only its invariants -- monotone decrease, fixed point -- are tested).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
#define PI_L 3.14159265358979323846264338327950288419716939937510L

/* ------------------------------------------------------------------------------------------------
 * O1 geometry: HEALPix RING scheme (paper: "HEALPix pixelization"; reading G3).
 * Rings i = 1 .. 4 nside - 1, north to south.
 *   north cap  1 <= i < nside      : N_i = 4 i,     z_i = 1 - i^2/(3 nside^2),     phi0 = pi/(4 i)
 *   belt       nside <= i <= 3nside: N_i = 4 nside, z_i = 4/3 - 2 i/(3 nside),
 *                                    phi0 = pi/(4 nside) if (i - nside) even else 0
 *   south cap  mirror of ring 4 nside - i (same N, same phi0, z -> -z).
 * phi0 is always shift * pi / N_i with shift in {0,1}; this is what is returned, so that every phase
 * m (phi0 + 2 pi n / N) = 2 pi (m shift + 2 m n) / (2 N) can be reduced in integers.
 * omz = 1 - |z| is returned separately so that sin^2(theta) = omz (2 - omz) has no cancellation.
 * ---------------------------------------------------------------------------------------------- */
typedef struct { long long n, start; int shift; ld z, sin2; } ring_t;

static ring_t ring_info(int nside, int i)
{
    ring_t r;
    long long ns = nside;
    int south = (i > 2 * nside);
    long long j = south ? 4 * ns - i : i;            /* mirror ring in the north (or equator) */
    ld absz;
    if (j < ns) {                                    /* polar cap */
        r.n = 4 * j;
        ld omz = (ld)(j * j) / (ld)(3 * ns * ns);
        absz = 1.0L - omz;
        r.sin2 = omz * (2.0L - omz);
        r.shift = 1;
        r.start = 2 * j * (j - 1);                   /* sum_{t<j} 4t */
    } else {                                         /* equatorial belt */
        r.n = 4 * ns;
        absz = (ld)(4 * ns - 2 * j) / (ld)(3 * ns);
        r.sin2 = (1.0L - absz) * (1.0L + absz);
        r.shift = ((j - ns) % 2 == 0) ? 1 : 0;
        r.start = 2 * ns * (ns - 1) + (j - ns) * 4 * ns;
    }
    if (south) {
        long long npix = 12 * ns * ns;
        r.start = npix - r.start - r.n;              /* mirrored position */
        r.z = -absz;
    } else {
        r.z = absz;
    }
    return r;
}

long long oracle_npix(int nside) { return 12LL * nside * nside; }
long long oracle_nalm(int lmax) { return (long long)(lmax + 1) * (lmax + 2) / 2; }
long long oracle_alm_index(int lmax, int l, int m) { return (long long)m * (2 * lmax + 1 - m) / 2 + l; }
int oracle_nrings(int nside) { return 4 * nside - 1; }
int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ring i (1-based): number of pixels, first pixel, z = cos(theta), phi0 (as double, for tests) */
void oracle_ring_info(int nside, int i, long long* n, long long* start, double* z, double* phi0)
{
    ring_t r = ring_info(nside, i);
    *n = r.n; *start = r.start; *z = (double)r.z;
    *phi0 = (double)(r.shift * PI_L / (ld)r.n);
}

/* ------------------------------------------------------------------------------------------------
 * O2 normalised associated Legendre functions lambda_lm (PAPER.md:82 fn. 2: |P_l^m| = |Y_lm|;
 * reading G2: orthonormal Y_lm = lambda_lm(theta) e^{i m phi} with the Condon-Shortley phase).
 *   seed       lambda_mm = (-1)^m sqrt((2m+1)/(4 pi) (2m-1)!!/(2m)!!) sin^m(theta)
 *   recurrence lambda_lm = a_lm (z lambda_{l-1,m} - b_lm lambda_{l-2,m}),
 *              a_lm = sqrt((4 l^2 - 1)/(l^2 - m^2)),  b_lm = sqrt(((l-1)^2 - m^2)/(4 (l-1)^2 - 1)).
 * The pair (cur, prev) is carried as long double mantissas times 2^e with an explicit integer
 * exponent e, so the seed sin^m(theta) can be as small as it likes (paper item 11, PAPER.md:230-232,
 * describes why a plain 64-bit recurrence underflows; the oracle simply never does).
 * coef = table of (a_lm, b_lm) for this m, l = m..lmax (entries l = m unused).
 * out[l - m] = lambda_lm as long double (0 only if the true value is below ~1e-4900).
 * ---------------------------------------------------------------------------------------------- */
static void lambda_coef(int lmax, int m, ld* a, ld* b)
{
    for (int l = m + 1; l <= lmax; ++l) {
        ld l2 = (ld)l * l, m2 = (ld)m * m, lm1 = (ld)(l - 1) * (l - 1);
        a[l - m] = sqrtl((4.0L * l2 - 1.0L) / (l2 - m2));
        b[l - m] = sqrtl((lm1 - m2) / (4.0L * lm1 - 1.0L));
    }
    a[0] = b[0] = 0.0L;
}

static void lambda_lm(int lmax, int m, ld z, ld sin2, const ld* a, const ld* b, ld* out)
{
    /* log2 |lambda_mm| */
    ld lg = 0.5L * log2l((2.0L * m + 1.0L) / (4.0L * PI_L));
    for (int j = 1; j <= m; ++j) lg += 0.5L * log2l((ld)(2 * j - 1) / (ld)(2 * j));
    if (m > 0) {
        if (sin2 <= 0.0L) { for (int l = m; l <= lmax; ++l) out[l - m] = 0.0L; return; }
        lg += 0.5L * (ld)m * log2l(sin2);
    }
    ld fl = floorl(lg);
    long e = (long)fl;
    ld cur = exp2l(lg - fl);                         /* mantissa in [1,2) */
    if (m & 1) cur = -cur;
    ld prev = 0.0L;
    const long BIG = 8000;
    const ld big = ldexpl(1.0L, (int)BIG), inv_big = ldexpl(1.0L, -(int)BIG);
    out[0] = ldexpl(cur, (int)(e < -40000 ? -40000 : e));
    for (int l = m + 1; l <= lmax; ++l) {
        ld nxt = a[l - m] * (z * cur - b[l - m] * prev);
        prev = cur; cur = nxt;
        if (fabsl(cur) > big) { cur *= inv_big; prev *= inv_big; e += BIG; }
        out[l - m] = ldexpl(cur, (int)(e < -40000 ? -40000 : e));
    }
}

/* test entry: lambda_lm(z) for l = m..lmax at an arbitrary z = cos(theta), double in / double out */
void oracle_lambda(int lmax, int m, double z, double* out)
{
    int n = lmax - m + 1;
    ld* a = (ld*)malloc(sizeof(ld) * n); ld* b = (ld*)malloc(sizeof(ld) * n); ld* o = (ld*)malloc(sizeof(ld) * n);
    lambda_coef(lmax, m, a, b);
    ld zl = (ld)z;
    lambda_lm(lmax, m, zl, (1.0L - zl) * (1.0L + zl), a, b, o);
    for (int i = 0; i < n; ++i) out[i] = (double)o[i];
    free(a); free(b); free(o);
}

/* test entry: lambda_lm on ring i of the nside grid, returned as (mantissa, exponent) pairs with
 * value = mant * 2^expo, so that values far below the double range can still be inspected */
void oracle_lambda_ring(int nside, int iring, int lmax, int m, double* mant, int* expo)
{
    int n = lmax - m + 1;
    ld* a = (ld*)malloc(sizeof(ld) * n); ld* b = (ld*)malloc(sizeof(ld) * n); ld* o = (ld*)malloc(sizeof(ld) * n);
    lambda_coef(lmax, m, a, b);
    ring_t r = ring_info(nside, iring);
    lambda_lm(lmax, m, r.z, r.sin2, a, b, o);
    for (int i = 0; i < n; ++i) { int ex; ld mt = frexpl(o[i], &ex); mant[i] = (double)mt; expo[i] = ex; }
    free(a); free(b); free(o);
}

/* ------------------------------------------------------------------------------------------------
 * O5 spin-2 functions (eq. 8, 125-127 eq. 12, 449 eq. A5: F+ = -X1, F- = -X2 with
 * X1 = (+2Y + -2Y)/2, X2 = (+2Y - -2Y)/2 without the e^{i m phi} factor; spin-weighted harmonics of
 * Zaldarriaga & Seljak, the paper's reference at PAPER.md:103).  Closed form, l >= 2, x = cos(theta):
 *   N_l  = 2 / sqrt((l-1) l (l+1) (l+2)),   c_lm = sqrt((2l+1)/(2l-1) (l^2 - m^2))
 *   X1 = N_l { -[(l - m^2)/sin^2 + l(l-1)/2] lambda_lm + (x/sin^2) c_lm lambda_{l-1,m} }
 *   X2 = N_l (m/sin^2) { c_lm lambda_{l-1,m} - (l-1) x lambda_lm }
 * lam[l-m] as produced by lambda_lm; x1/x2[l-m] written for l = max(m,2)..lmax, 0 below l = 2.
 * ---------------------------------------------------------------------------------------------- */
static void spin2_x(int lmax, int m, ld z, ld sin2, const ld* lam, ld* x1, ld* x2)
{
    for (int l = m; l <= lmax; ++l) {
        if (l < 2) { x1[l - m] = x2[l - m] = 0.0L; continue; }
        ld L = (ld)l, M = (ld)m;
        ld nl = 2.0L / sqrtl((L - 1.0L) * L * (L + 1.0L) * (L + 2.0L));
        ld clm = sqrtl((2.0L * L + 1.0L) / (2.0L * L - 1.0L) * (L * L - M * M));
        ld lam_l = lam[l - m];
        ld lam_lm1 = (l > m) ? lam[l - 1 - m] : 0.0L;
        x1[l - m] = nl * (-((L - M * M) / sin2 + 0.5L * L * (L - 1.0L)) * lam_l + (z / sin2) * clm * lam_lm1);
        x2[l - m] = nl * (M / sin2) * (clm * lam_lm1 - (L - 1.0L) * z * lam_l);
    }
}

/* test entry: X1, X2 at arbitrary z for l = m..lmax */
void oracle_spin2_x(int lmax, int m, double z, double* x1, double* x2)
{
    int n = lmax - m + 1;
    ld* a = (ld*)malloc(sizeof(ld) * n); ld* b = (ld*)malloc(sizeof(ld) * n);
    ld* o = (ld*)malloc(sizeof(ld) * n); ld* p = (ld*)malloc(sizeof(ld) * n); ld* q = (ld*)malloc(sizeof(ld) * n);
    lambda_coef(lmax, m, a, b);
    ld zl = (ld)z, s2 = (1.0L - zl) * (1.0L + zl);
    lambda_lm(lmax, m, zl, s2, a, b, o);
    spin2_x(lmax, m, zl, s2, o, p, q);
    for (int i = 0; i < n; ++i) { x1[i] = (double)p[i]; x2[i] = (double)q[i]; }
    free(a); free(b); free(o); free(p); free(q);
}

/* ------------------------------------------------------------------------------------------------
 * Phase tables.  For a ring of N pixels every phase that occurs is 2 pi j / (2N), j integer
 * (see ring_info).  tab_c/tab_s[j] = cos/sin(pi j / N), j = 0 .. 2N-1, one table per distinct N.
 * This is a lookup of exactly reduced phases, not an FFT.
 * ---------------------------------------------------------------------------------------------- */
typedef struct { int nside; ld** c; ld** s; } phase_tabs;     /* indexed by N/4 = 1..nside */

static void phase_tabs_build(phase_tabs* t, int nside)
{
    t->nside = nside;
    t->c = (ld**)calloc(nside + 1, sizeof(ld*));
    t->s = (ld**)calloc(nside + 1, sizeof(ld*));
    #pragma omp parallel for schedule(dynamic, 4)
    for (int q = 1; q <= nside; ++q) {
        long long N = 4LL * q;
        t->c[q] = (ld*)malloc(sizeof(ld) * 2 * N);
        t->s[q] = (ld*)malloc(sizeof(ld) * 2 * N);
        for (long long j = 0; j < 2 * N; ++j) {
            ld ang = PI_L * (ld)j / (ld)N;
            t->c[q][j] = cosl(ang); t->s[q][j] = sinl(ang);
        }
    }
}
static void phase_tabs_free(phase_tabs* t)
{
    for (int q = 1; q <= t->nside; ++q) { free(t->c[q]); free(t->s[q]); }
    free(t->c); free(t->s);
}

/* ring Fourier sum of eq. 2:
 *   T_m(theta_i) = dsigma * sum_n T(i,n) exp(-i m (phi0_i + 2 pi n / N_i))
 * evaluated term by term with the phase index (m shift + 2 m n) mod 2N. */
static void ring_fourier(const double* pix, const ring_t* r, int m, const ld* tc, const ld* ts,
                         ld dsigma, ld* re, ld* im)
{
    long long N2 = 2 * r->n;
    long long idx = ((long long)m * r->shift) % N2;
    long long step = (2LL * m) % N2;
    ld sr = 0.0L, si = 0.0L;
    for (long long n = 0; n < r->n; ++n) {
        ld t = (ld)pix[n];
        sr += t * tc[idx];
        si -= t * ts[idx];
        idx += step; if (idx >= N2) idx -= N2;
    }
    *re = sr * dsigma; *im = si * dsigma;
}

/* ------------------------------------------------------------------------------------------------
 * O3 analysis (eq. 1-2; Alg. 1; readings G1, G4, G5, G7):
 *   a_lm^k = sum_i lambda_lm(theta_i) T_m^k(theta_i),   0 <= m <= l <= lmax,  dsigma = 4 pi / npix.
 * spin 2 (eq. 14 with F+ = -X1, F- = -X2; reading O5):
 *   a_E = - sum_i [ X1 Q_m + i X2 U_m ],   a_B = - sum_i [ X1 U_m - i X2 Q_m ].
 * mlist/nm: the m values to compute (NULL -> all 0..lmax).  Entries of other m are left untouched.
 * Im(a_l0) is written as exactly 0; spin-2 entries with l < 2 are written as 0.
 * ---------------------------------------------------------------------------------------------- */
void oracle_analysis(int nside, int lmax, int nmaps, int spin, const double* maps, double* alm,
                     const int* mlist, int nm)
{
    const int ncomp = (spin == 2) ? 2 : 1;
    const long long npix = oracle_npix(nside), nalm = oracle_nalm(lmax);
    const int nrings = 4 * nside - 1;
    const ld dsigma = 4.0L * PI_L / (ld)npix;
    phase_tabs tabs; phase_tabs_build(&tabs, nside);
    int all = (mlist == NULL);
    if (all) nm = lmax + 1;

    #pragma omp parallel for schedule(dynamic, 1)
    for (int im = 0; im < nm; ++im) {
        const int m = all ? im : mlist[im];
        const int nl = lmax - m + 1;
        ld* a = (ld*)malloc(sizeof(ld) * nl); ld* b = (ld*)malloc(sizeof(ld) * nl);
        ld* lam = (ld*)malloc(sizeof(ld) * nl);
        ld* x1 = (ld*)malloc(sizeof(ld) * nl); ld* x2 = (ld*)malloc(sizeof(ld) * nl);
        /* accumulators [map][comp][l][re,im] */
        ld* acc = (ld*)calloc((size_t)nmaps * ncomp * nl * 2, sizeof(ld));
        lambda_coef(lmax, m, a, b);
        for (int i = 1; i <= nrings; ++i) {
            ring_t r = ring_info(nside, i);
            const ld* tc = tabs.c[r.n / 4]; const ld* ts = tabs.s[r.n / 4];
            lambda_lm(lmax, m, r.z, r.sin2, a, b, lam);
            if (spin == 2) spin2_x(lmax, m, r.z, r.sin2, lam, x1, x2);
            for (int k = 0; k < nmaps; ++k) {
                if (spin != 2) {
                    ld tr, ti;
                    ring_fourier(maps + (size_t)k * npix + r.start, &r, m, tc, ts, dsigma, &tr, &ti);
                    ld* ac = acc + (size_t)k * nl * 2;
                    for (int l = m; l <= lmax; ++l) {
                        ac[2 * (l - m)] += lam[l - m] * tr;
                        ac[2 * (l - m) + 1] += lam[l - m] * ti;
                    }
                } else {
                    ld qr, qi, ur, ui;
                    ring_fourier(maps + ((size_t)k * 2 + 0) * npix + r.start, &r, m, tc, ts, dsigma, &qr, &qi);
                    ring_fourier(maps + ((size_t)k * 2 + 1) * npix + r.start, &r, m, tc, ts, dsigma, &ur, &ui);
                    ld* ae = acc + ((size_t)k * 2 + 0) * nl * 2;
                    ld* ab = acc + ((size_t)k * 2 + 1) * nl * 2;
                    for (int l = m; l <= lmax; ++l) {
                        ld p = x1[l - m], q = x2[l - m];
                        /* a_E = -(X1 Q + i X2 U):  i (ur + i ui) = -ui + i ur */
                        ae[2 * (l - m)]     -= p * qr - q * ui;
                        ae[2 * (l - m) + 1] -= p * qi + q * ur;
                        /* a_B = -(X1 U - i X2 Q): -i (qr + i qi) = qi - i qr */
                        ab[2 * (l - m)]     -= p * ur + q * qi;
                        ab[2 * (l - m) + 1] -= p * ui - q * qr;
                    }
                }
            }
        }
        for (int k = 0; k < nmaps; ++k)
            for (int c = 0; c < ncomp; ++c) {
                const ld* ac = acc + ((size_t)k * ncomp + c) * nl * 2;
                double* out = alm + (((size_t)k * ncomp + c) * nalm + oracle_alm_index(lmax, 0, m)) * 2;
                for (int l = m; l <= lmax; ++l) {
                    double re = (double)ac[2 * (l - m)], imv = (double)ac[2 * (l - m) + 1];
                    if (m == 0) imv = 0.0;
                    if (spin == 2 && l < 2) { re = 0.0; imv = 0.0; }
                    out[2 * l] = re; out[2 * l + 1] = imv;
                }
            }
        free(a); free(b); free(lam); free(x1); free(x2); free(acc);
    }
    phase_tabs_free(&tabs);
}

/* ------------------------------------------------------------------------------------------------
 * O4 synthesis (eq. 4-5; readings G7, G8):
 *   T^k(i,n) = sum_{m=0}^{lmax} w_m Re[ (sum_{l=m}^{lmax} a_lm^k lambda_lm(theta_i)) e^{+i m (phi0_i + 2 pi n/N_i)} ],
 *   w_0 = 1, w_{m>0} = 2 (the m<0 half of eq. 4's sum, with a_{l,-m} = (-1)^m conj(a_lm)); Im(a_l0) ignored.
 * spin 2 (eq. 15; reading O5):
 *   q_m = - sum_l [ a_E X1 + i a_B X2 ],  u_m = - sum_l [ a_B X1 - i a_E X2 ],
 *   Q = sum_m w_m Re[q_m e^{i m phi}],  U likewise;  entries with l < 2 ignored.
 * rlist/nr: rings (1-based) to compute (NULL -> all).  Pixels of other rings are left untouched.
 * ---------------------------------------------------------------------------------------------- */
void oracle_synthesis(int nside, int lmax, int nmaps, int spin, const double* alm, double* maps,
                      const int* rlist, int nr)
{
    const int ncomp = (spin == 2) ? 2 : 1;
    const long long npix = oracle_npix(nside), nalm = oracle_nalm(lmax);
    const int nrings = 4 * nside - 1;
    phase_tabs tabs; phase_tabs_build(&tabs, nside);
    /* recurrence coefficients for every (l,m), m-major like the alm index */
    ld* ca = (ld*)malloc(sizeof(ld) * nalm); ld* cb = (ld*)malloc(sizeof(ld) * nalm);
    #pragma omp parallel for schedule(dynamic, 8)
    for (int m = 0; m <= lmax; ++m) {
        long long o = oracle_alm_index(lmax, m, m);
        lambda_coef(lmax, m, ca + o, cb + o);
    }
    int all = (rlist == NULL);
    if (all) nr = nrings;

    #pragma omp parallel for schedule(dynamic, 1)
    for (int ir = 0; ir < nr; ++ir) {
        const int i = all ? ir + 1 : rlist[ir];
        ring_t r = ring_info(nside, i);
        const ld* tc = tabs.c[r.n / 4]; const ld* ts = tabs.s[r.n / 4];
        const long long N = r.n, N2 = 2 * N;
        ld* lam = (ld*)malloc(sizeof(ld) * (lmax + 1));
        ld* x1 = (ld*)malloc(sizeof(ld) * (lmax + 1)); ld* x2 = (ld*)malloc(sizeof(ld) * (lmax + 1));
        ld* pix = (ld*)calloc((size_t)nmaps * ncomp * N, sizeof(ld));
        for (int m = 0; m <= lmax; ++m) {
            long long o = oracle_alm_index(lmax, m, m);
            lambda_lm(lmax, m, r.z, r.sin2, ca + o, cb + o, lam);
            if (spin == 2) spin2_x(lmax, m, r.z, r.sin2, lam, x1, x2);
            const ld w = (m == 0) ? 1.0L : 2.0L;
            for (int k = 0; k < nmaps; ++k) {
                ld fr[2], fi[2];                      /* per component: T_m (or q_m, u_m) */
                if (spin != 2) {
                    const double* a = alm + ((size_t)k * nalm + oracle_alm_index(lmax, 0, m)) * 2;
                    ld sr = 0.0L, si = 0.0L;
                    for (int l = m; l <= lmax; ++l) {
                        sr += (ld)a[2 * l] * lam[l - m];
                        if (m > 0) si += (ld)a[2 * l + 1] * lam[l - m];
                    }
                    fr[0] = sr; fi[0] = si;
                } else {
                    const double* ae = alm + (((size_t)k * 2 + 0) * nalm + oracle_alm_index(lmax, 0, m)) * 2;
                    const double* ab = alm + (((size_t)k * 2 + 1) * nalm + oracle_alm_index(lmax, 0, m)) * 2;
                    ld qr = 0, qi = 0, ur = 0, ui = 0;
                    for (int l = (m > 2 ? m : 2); l <= lmax; ++l) {
                        ld er = ae[2 * l], ei = (m > 0) ? (ld)ae[2 * l + 1] : 0.0L;
                        ld br = ab[2 * l], bi = (m > 0) ? (ld)ab[2 * l + 1] : 0.0L;
                        ld p = x1[l - m], q = x2[l - m];
                        /* q_m = -(a_E X1 + i a_B X2) */
                        qr -= er * p - bi * q;
                        qi -= ei * p + br * q;
                        /* u_m = -(a_B X1 - i a_E X2) */
                        ur -= br * p + ei * q;
                        ui -= bi * p - er * q;
                    }
                    fr[0] = qr; fi[0] = qi; fr[1] = ur; fi[1] = ui;
                }
                for (int c = 0; c < ncomp; ++c) {
                    ld* p = pix + ((size_t)k * ncomp + c) * N;
                    long long idx = ((long long)m * r.shift) % N2;
                    long long step = (2LL * m) % N2;
                    for (long long n = 0; n < N; ++n) {
                        /* Re[(fr + i fi)(cos + i sin)] */
                        p[n] += w * (fr[c] * tc[idx] - fi[c] * ts[idx]);
                        idx += step; if (idx >= N2) idx -= N2;
                    }
                }
            }
        }
        for (int k = 0; k < nmaps; ++k)
            for (int c = 0; c < ncomp; ++c) {
                double* out = maps + ((size_t)k * ncomp + c) * npix + r.start;
                const ld* p = pix + ((size_t)k * ncomp + c) * N;
                for (long long n = 0; n < N; ++n) out[n] = (double)p[n];
            }
        free(lam); free(x1); free(x2); free(pix);
    }
    free(ca); free(cb);
    phase_tabs_free(&tabs);
}

/* ------------------------------------------------------------------------------------------------
 * O6 iterative analysis, "traditional" scheme (Alg. 2; "the mode adopted
 * by HEALPix, a_lm updated outside the m-loop"; readings G16, G17, G18):
 *   a(0) = analysis(map);  for n = 0..niter-1:  r(n) = map - synthesis(a(n));
 *   rms(n)_k = sqrt(mean_pixels r(n)_k^2);  a(n+1) = a(n) + analysis(r(n)).
 * Done in pixel space (the CUDA path does it between T_m and a_lm; that the two agree is the paper's
 * "FFT is lossless" claim).  resid_rms: [niter][nmaps*ncomp] or NULL.
 * ---------------------------------------------------------------------------------------------- */
void oracle_analysis_iter(int nside, int lmax, int nmaps, int spin, const double* maps, double* alm,
                          int niter, double* resid_rms)
{
    const int ncomp = (spin == 2) ? 2 : 1;
    const long long npix = oracle_npix(nside), nalm = oracle_nalm(lmax);
    const size_t nmap_tot = (size_t)nmaps * ncomp * npix, nalm_tot = (size_t)nmaps * ncomp * nalm * 2;
    oracle_analysis(nside, lmax, nmaps, spin, maps, alm, NULL, 0);
    double* res = (double*)malloc(sizeof(double) * nmap_tot);
    double* da = (double*)calloc(nalm_tot, sizeof(double));
    for (int it = 0; it < niter; ++it) {
        oracle_synthesis(nside, lmax, nmaps, spin, alm, res, NULL, 0);
        for (size_t p = 0; p < nmap_tot; ++p) res[p] = maps[p] - res[p];
        if (resid_rms)
            for (int kc = 0; kc < nmaps * ncomp; ++kc) {
                ld s = 0.0L;
                for (long long p = 0; p < npix; ++p) { ld v = res[(size_t)kc * npix + p]; s += v * v; }
                resid_rms[(size_t)it * nmaps * ncomp + kc] = (double)sqrtl(s / (ld)npix);
            }
        oracle_analysis(nside, lmax, nmaps, spin, res, da, NULL, 0);
        for (size_t q = 0; q < nalm_tot; ++q) alm[q] += da[q];
    }
    free(res); free(da);
}
