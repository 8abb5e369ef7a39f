/* Driver for tests/test_oracle_sanitize.py: calls every exported routine of oracle/sht_oracle.c on tiny inputs (ragged:
 * nside 3 and 4, lmax 8 and 11, spin 0 and 2, restricted m / ring lists), compiled together with the oracle under
 * -fsanitize=address,undefined.  It checks nothing about the values beyond "finite and not all zero" -- the pins in
 * tests/test_oracle_*.py do that; this run is about out-of-bounds accesses, uninitialised-size arithmetic and undefined
 * behaviour inside the oracle.  Test infrastructure: includes nothing of the product. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

long long oracle_npix(int nside);
long long oracle_nalm(int lmax);
long long oracle_alm_index(int lmax, int l, int m);
int oracle_nrings(int nside);
int oracle_num_threads(void);
void oracle_ring_info(int nside, int i, long long* n, long long* start, double* z, double* phi0);
void oracle_lambda(int lmax, int m, double z, double* out);
void oracle_lambda_ring(int nside, int iring, int lmax, int m, double* mant, int* expo);
void oracle_spin2_x(int lmax, int m, double z, double* x1, double* x2);
void oracle_analysis(int nside, int lmax, int nmaps, int spin, const double* maps, double* alm, const int* mlist, int nm);
void oracle_synthesis(int nside, int lmax, int nmaps, int spin, const double* alm, double* maps, const int* rlist, int nr);
void oracle_analysis_iter(int nside, int lmax, int nmaps, int spin, const double* maps, double* alm, int niter, double* resid_rms);

static unsigned long long state = 88172645463325252ULL;
static double rnd(void)
{
    state ^= state << 13; state ^= state >> 7; state ^= state << 17;
    return (double)(state >> 11) / 9007199254740992.0 - 0.5;
}

static int finite_nonzero(const double* x, long long n, const char* what)
{
    double s = 0.0;
    for (long long i = 0; i < n; ++i) {
        if (!isfinite(x[i])) { fprintf(stderr, "%s: entry %lld is not finite\n", what, i); return 0; }
        s += fabs(x[i]);
    }
    if (s == 0.0) { fprintf(stderr, "%s: all zero\n", what); return 0; }
    return 1;
}

static int run(int nside, int lmax, int nmaps, int spin)
{
    const int ncomp = spin == 2 ? 2 : 1;
    const long long npix = oracle_npix(nside), nalm = oracle_nalm(lmax);
    /* exactly sized buffers: one element too few anywhere is an ASan report */
    double* alm = malloc(sizeof(double) * 2 * nalm * ncomp * nmaps);
    double* alm2 = malloc(sizeof(double) * 2 * nalm * ncomp * nmaps);
    double* maps = malloc(sizeof(double) * npix * ncomp * nmaps);
    double* rms = malloc(sizeof(double) * 3 * ncomp * nmaps);
    int ok = alm && alm2 && maps && rms;
    if (!ok) return 0;
    for (long long i = 0; i < 2 * nalm * ncomp * nmaps; ++i) alm[i] = rnd();
    oracle_synthesis(nside, lmax, nmaps, spin, alm, maps, NULL, 0);
    ok = ok && finite_nonzero(maps, npix * ncomp * nmaps, "synthesis");
    int rlist[3] = {1, 2 * nside, 4 * nside - 1};                  /* first, equator and last ring */
    oracle_synthesis(nside, lmax, nmaps, spin, alm, maps, rlist, 3);
    for (long long i = 0; i < npix * ncomp * nmaps; ++i) maps[i] += 0.01 * rnd();
    oracle_analysis(nside, lmax, nmaps, spin, maps, alm2, NULL, 0);
    ok = ok && finite_nonzero(alm2, 2 * nalm * ncomp * nmaps, "analysis");
    int mlist[3] = {0, lmax / 2, lmax};
    oracle_analysis(nside, lmax, nmaps, spin, maps, alm2, mlist, 3);
    oracle_analysis_iter(nside, lmax, nmaps, spin, maps, alm2, 3, rms);
    ok = ok && finite_nonzero(alm2, 2 * nalm * ncomp * nmaps, "analysis_iter") && finite_nonzero(rms, 3 * ncomp * nmaps, "rms");
    oracle_analysis_iter(nside, lmax, nmaps, spin, maps, alm2, 0, NULL);
    free(alm); free(alm2); free(maps); free(rms);
    return ok;
}

int main(void)
{
    int ok = 1;
    if (oracle_npix(4) != 192 || oracle_nalm(11) != 78 || oracle_alm_index(11, 11, 11) != 77 || oracle_nrings(4) != 15) ok = 0;
    if (oracle_num_threads() < 1) ok = 0;
    for (int nside = 1; nside <= 5; ++nside) {
        long long total = 0;
        for (int i = 1; i <= 4 * nside - 1; ++i) {
            long long n, start; double z, phi0;
            oracle_ring_info(nside, i, &n, &start, &z, &phi0);
            if (start != total || n < 4 || fabs(z) >= 1.0) ok = 0;
            total += n;
        }
        if (total != oracle_npix(nside)) ok = 0;
    }
    for (int lmax = 2; lmax <= 40; lmax += 19) {
        for (int m = 0; m <= lmax; m += (lmax > 4 ? lmax / 4 : 1)) {
            const int n = lmax - m + 1;
            double* out = malloc(sizeof(double) * n);
            double* x1 = malloc(sizeof(double) * n);
            double* x2 = malloc(sizeof(double) * n);
            int* ex = malloc(sizeof(int) * n);
            oracle_lambda(lmax, m, 0.3, out);
            oracle_lambda(lmax, m, -1.0, out);                       /* the poles: sin = 0 */
            oracle_lambda(lmax, m, 1.0, out);
            oracle_spin2_x(lmax, m, 0.3, x1, x2);
            oracle_lambda_ring(4, 1, lmax, m, out, ex);
            oracle_lambda_ring(4, 8, lmax, m, out, ex);
            free(out); free(x1); free(x2); free(ex);
        }
    }
    ok = ok && run(4, 11, 3, 0);
    ok = ok && run(3, 8, 2, 0);
    ok = ok && run(4, 11, 2, 2);
    ok = ok && run(3, 7, 1, 2);
    ok = ok && run(1, 2, 1, 0);
    ok = ok && run(1, 2, 1, 2);
    printf(ok ? "oracle sanitize run: ok\n" : "oracle sanitize run: FAILED\n");
    return ok ? 0 : 1;
}
