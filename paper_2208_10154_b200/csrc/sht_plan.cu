// sht_plan.cu -- plan creation: ring tables, FFT twiddles / radix lists, recurrence coefficients and the
// l_safe / seed table of PAPER.md:230-232 (item 11: "the recursion starts from safe positions ... computed
// once and saved as an input table l_safe(m, theta)").
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <thread>
#include <utility>
#include <vector>
#include "sht_internal.h"

namespace sht {

// ------------------------------------------------------------------------------------------------
// Seed kernel.  One thread per (m, p).  lambda_mm = c_m sin^m(theta) is formed as a
// (mantissa, exponent) pair so that it cannot underflow, then the three-term recurrence
//   lambda_l = alpha_l z lambda_{l-1} - beta_l lambda_{l-2}
// is stepped with a shared power-of-two exponent until |lambda_l| >= 2^-70 (~8.5e-22, below the paper's
// example threshold 1e-20).  That l is l_safe(m,p); the two values before it are stored as plain doubles,
// so the hot kernels run an unscaled recurrence from there and treat lambda below l_safe as zero.
// ------------------------------------------------------------------------------------------------
constexpr int SEED_THRESH_EXP = -70;

__device__ inline void renorm(double& f, int& e)
{
    int t;
    f = frexp(f, &t);
    e += t;
}

__global__ void k_seed_table(DevicePlan d, const double* __restrict__ cm, int* __restrict__ lstart,
                             double2* __restrict__ seed)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)(d.lmax + 1) * d.nh;
    if (gid >= total) return;
    const int m = (int)(gid / d.nh), p = (int)(gid % d.nh);
    const double z = d.z[p];
    // sin^m(theta) by binary powering on (mantissa, exponent)
    double bf; int be;
    bf = frexp(sqrt(d.sin2[p]), &be);
    double rf = 1.0; int re = 0;
    for (int n = m; n > 0; n >>= 1) {
        if (n & 1) { rf *= bf; re += be; renorm(rf, re); }
        bf *= bf; be *= 2; renorm(bf, be);
    }
    double cur = cm[m] * rf; int E = re;
    renorm(cur, E);                              // lambda_mm = cur * 2^E, |cur| in [0.5, 1)
    double prev = 0.0, prev2 = 0.0;
    int ls = d.lmax + 1;
    double x1 = 0.0, x2 = 0.0;
    if (ilogb(cur) + E >= SEED_THRESH_EXP) {
        ls = m; x1 = 0.0; x2 = ldexp(cur, E);    // coef(l = m) = (0, -1) reproduces lambda_mm = x2
    } else {
        const double2* cf = d.coef + ((long long)m * (2 * d.lmax + 1 - m) / 2);
        for (int l = m + 1; l <= d.lmax; ++l) {
            const double2 ab = cf[l];
            const double nxt = ab.x * z * cur - ab.y * prev;
            prev2 = prev; prev = cur; cur = nxt;
            if (fabs(cur) > 0x1p200) { cur *= 0x1p-200; prev *= 0x1p-200; prev2 *= 0x1p-200; E += 200; }
            if (cur != 0.0 && ilogb(cur) + E >= SEED_THRESH_EXP) {
                ls = l; x1 = ldexp(prev, E); x2 = ldexp(prev2, E);
                break;
            }
        }
    }
    lstart[gid] = ls;
    seed[gid] = make_double2(x1, x2);
}

// Recurrence state at every LEG_CS-th l (DevicePlan::cseed): the same arithmetic, in the same order, as the
// generator warps of the Legendre kernels, so a chain restarted from a table entry reproduces the sequential chain
// bit for bit.
__global__ void k_chunk_seeds(DevicePlan d, double2* __restrict__ cseed)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)(d.lmax + 1) * d.nh;
    if (gid >= total) return;
    const int m = (int)(gid / d.nh), p = (int)(gid % d.nh);
    const double z = d.z[p];
    const double2 sd = d.seed[gid];
    double x1 = sd.x, x2 = sd.y;
    const int ls = d.lstart[gid];
    const double2* cf = d.coef + ((long long)m * (2 * d.lmax + 1 - m) / 2);
    double2* out = cseed + (size_t)d.csoff[m] * d.nh + p;
    for (int l = m; l <= d.lmax; ++l) {
        if (((l - m) & (LEG_CS - 1)) == 0) { *out = make_double2(x1, x2); out += d.nh; }
        if (l >= ls) {
            const double2 ab = cf[l];
            const double t = fma(ab.x * z, x1, -(ab.y * x2));
            x2 = x1; x1 = t;
        }
    }
}

cudaError_t launch_chunk_seeds(const DevicePlan& d, double2* cseed, cudaStream_t st)
{
    const long long total = (long long)(d.lmax + 1) * d.nh;
    const int bs = 128;
    k_chunk_seeds<<<(unsigned)((total + bs - 1) / bs), bs, 0, st>>>(d, cseed);
    return cudaGetLastError();
}

cudaError_t launch_seed_table(const DevicePlan& d, const double* cm, int* lstart, double2* seed, cudaStream_t st)
{
    const long long total = (long long)(d.lmax + 1) * d.nh;
    const int bs = 128;
    k_seed_table<<<(unsigned)((total + bs - 1) / bs), bs, 0, st>>>(d, cm, lstart, seed);
    return cudaGetLastError();
}

}  // namespace sht

using namespace sht;

// ------------------------------------------------------------------------------------------------
// host-side table construction
// ------------------------------------------------------------------------------------------------
static const long double PI_LD = 3.14159265358979323846264338327950288419716939937510L;

// Radix list of ring length n = 4 q in forward (analysis) order: primes >= 11 first (largest first; the first
// pass is fused with the global load, further ones run out of place), then 4s, a 2, and the 3s, 5s, 7s,
// which run in place.  The inverse transform (synthesis) walks the same list backwards.
static int factorize_ring(int n, std::vector<int>& out)
{
    std::vector<int> small, big;
    int r = n;
    while (r % 4 == 0) { small.push_back(4); r /= 4; }
    while (r % 2 == 0) { small.push_back(2); r /= 2; }
    for (int f = 3; (long long)f * f <= r; f += 2)
        while (r % f == 0) { (f <= 7 ? small : big).push_back(f); r /= f; }
    if (r > 1) (r <= 7 ? small : big).push_back(r);
    for (size_t i = big.size(); i-- > 0;) out.push_back(big[i]);
    for (int v : small) out.push_back(v);
    // primes 11 .. 31 run in place (register stages); only larger ones (rings too long for Bluestein) need two buffers
    int ngeneric = 0;
    for (int v : big) ngeneric += v >= BLUESTEIN_MIN_PRIME ? 1 : 0;
    return ngeneric;
}

template <typename T>
static cudaError_t upload(sht_plan_s* pl, const std::vector<T>& h, const T** dptr)
{
    void* p = nullptr;
    size_t bytes = h.size() * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) return e;
    pl->dev_allocs[pl->n_allocs++] = p;
    pl->table_bytes += bytes;
    if (!h.empty()) e = cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
    *dptr = (const T*)p;
    return e;
}

// plan-time FFT in long double (recursive decimation in time over the prime factors 2, 3, 5 of the length), for the
// Bluestein filter spectra; wr/wi = exp(-2 pi i e / N) of the top-level length N, this level has length N / stride
static void host_fft_rec(std::vector<long double>& re, std::vector<long double>& im, const std::vector<long double>& wr,
                         const std::vector<long double>& wi, size_t stride)
{
    const size_t n = re.size();
    if (n <= 1) return;
    size_t r = n;                                            // prime length: direct sum
    for (size_t f : {2, 3, 5, 7}) if (n % f == 0) { r = f; break; }
    const size_t mlen = n / r;
    std::vector<std::vector<long double>> sre(r, std::vector<long double>(mlen)), sim(r, std::vector<long double>(mlen));
    for (size_t q = 0; q < r; ++q)
        for (size_t j = 0; j < mlen; ++j) { sre[q][j] = re[j * r + q]; sim[q][j] = im[j * r + q]; }
    for (size_t q = 0; q < r; ++q) host_fft_rec(sre[q], sim[q], wr, wi, stride * r);
    for (size_t k = 0; k < n; ++k) {
        long double ar = 0.0L, ai = 0.0L;
        for (size_t q = 0; q < r; ++q) {
            const size_t e = ((q * k) % n) * stride;
            const long double xr = sre[q][k % mlen], xi = sim[q][k % mlen];
            ar += xr * wr[e] - xi * wi[e]; ai += xr * wi[e] + xi * wr[e];
        }
        re[k] = ar; im[k] = ai;
    }
}

static void host_fft(std::vector<long double>& re, std::vector<long double>& im)
{
    const size_t n = re.size();
    std::vector<long double> wr(n), wi(n);
    for (size_t e = 0; e < n; ++e) {
        const long double ang = -2.0L * PI_LD * (long double)e / (long double)n;
        wr[e] = cosl(ang); wi[e] = sinl(ang);
    }
    host_fft_rec(re, im, wr, wi, 1);
}

// convolution length of a Bluestein ring: the smallest of 2^a, 3 2^a, 5 2^a (a >= 2) that is >= minlen -- one odd
// pass at most, so the register-fused power-of-two passes keep doing the bulk of the work
static int bluestein_len(int minlen)
{
    int best = 0;
    for (int odd : {1, 3, 5}) {
        int v = 4 * odd;
        while (v < minlen) v *= 2;
        if (best == 0 || v < best) best = v;
    }
    return best;
}

// Kernel-side radix list: the power-of-two run of `f` (4s and at most one 2) is regrouped into register-fused
// passes, code 16 = two radix-4 stages, code 8 = a radix-4 and a radix-2 stage (grouped from the back, so that the
// last pass is the widest); other factors are copied.  The output order of the transform is unchanged, so the
// digit-reversal table is built from the plain list.
static void group_radices(const std::vector<int>& f, std::vector<int>& g)
{
    size_t i = 0;
    while (i < f.size()) {
        if (f[i] != 4 && f[i] != 2) { g.push_back(f[i]); ++i; continue; }
        int c4 = 0;
        while (i < f.size() && f[i] == 4) { ++c4; ++i; }
        const bool has2 = i < f.size() && f[i] == 2;
        if (has2) ++i;
        int pairable = c4 - ((has2 && c4 > 0) ? 1 : 0);
        if (pairable & 1) { g.push_back(4); --pairable; }
        for (int q = 0; q < pairable / 2; ++q) g.push_back(16);
        if (has2) g.push_back(c4 > 0 ? 8 : 2);
    }
}

// shared-memory padding shift of a pure power-of-two transform whose last pass is a fused 16 / 8 (31 = no padding)
static int pad_shift(const std::vector<int>& g, bool pure_pow2)
{
    if (!pure_pow2 || g.empty()) return 31;
    return g.back() == 16 ? 4 : g.back() == 8 ? 3 : 31;
}

// maps per CTA of the ring kernels: the largest power of two <= 16 whose buffers stay within 72 KB (two or three
// CTAs per SM); at least 2 maps (whole 32-byte sectors of the workspace lines) if that still fits one CTA per SM
static int ring_kt(size_t bytes_per_map)
{
    int kt = 1;
    while (kt * 2 <= 16 && (size_t)(kt * 2) * bytes_per_map <= (size_t)72 * 1024) kt *= 2;
    if (kt < 2 && 2 * bytes_per_map <= (size_t)224 * 1024) kt = 2;
    return kt;
}

extern "C" sht_status_t sht_plan_create(sht_plan_t* out, int nside, int lmax, int nmaps, int spin)
{
    return sht_plan_create_ex(out, nside, lmax, nmaps, spin, 0);
}

extern "C" sht_status_t sht_plan_create_ex(sht_plan_t* out, int nside, int lmax, int nmaps, int spin, size_t workspace_limit)
{
    if (!out) return SHT_ERR_NULL;
    *out = nullptr;
    if (nside < 1 || nside > 2048 || lmax < 0 || nmaps < 1 || (spin != 0 && spin != 2)) return SHT_ERR_INVALID_ARG;
    if (spin == 2 && lmax < 2) return SHT_ERR_INVALID_ARG;
    if (lmax > 16383) return SHT_ERR_UNSUPPORTED;

    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev == 0) return SHT_ERR_CUDA;      // no CPU fallback

    sht_plan_s* pl = (sht_plan_s*)calloc(1, sizeof(sht_plan_s));
    if (!pl) return SHT_ERR_ALLOC;
    DevicePlan& d = pl->d;
    d.nside = nside; d.lmax = lmax; d.spin = spin; d.ncomp = spin == 2 ? 2 : 1;
    d.nh = 2 * nside;
    d.npix = 12LL * nside * nside;
    d.nalm = (long long)(lmax + 1) * (lmax + 2) / 2;
    pl->nmaps = nmaps;

    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, dev);
    pl->sm_count = prop.multiProcessorCount;
    // ---- ring pairs, twiddles, radix lists ----------------------------------------------------
    std::vector<RingPair> rings(d.nh);
    std::vector<double> zs(d.nh), sin2s(d.nh);
    std::vector<double2> tw;
    std::vector<int> radix;
    std::vector<unsigned short> perm;
    std::vector<int> perm_off_of_q(nside + 1, 0), lc_of_q(nside + 1, 0), hf_off_of_q(nside + 1, 0);
    std::map<int, int> pow2_tw_off, pow2_fac_off, pow2_nfac;
    std::vector<int> tw_off_of_q(nside + 1, -1), fac_off_of_q(nside + 1, -1), nfac_of_q(nside + 1, 0), nbig_of_q(nside + 1, 0);
    std::vector<int> psh_of_q(nside + 1, 31);
    std::map<int, int> pow2_psh;
    for (int q = 1; q <= nside; ++q) {
        const int n = 4 * q;
        tw_off_of_q[q] = (int)tw.size();
        for (int j = 0; j < 2 * n; ++j) {
            long double ang = PI_LD * (long double)j / (long double)n;
            tw.push_back(make_double2((double)cosl(ang), (double)-sinl(ang)));
        }
        std::vector<int> f;
        nbig_of_q[q] = factorize_ring(n, f);
        if ((int)f.size() > MAX_RADIX_LIST) { free(pl); return SHT_ERR_UNSUPPORTED; }
        {
            std::vector<int> g;
            group_radices(f, g);
            fac_off_of_q[q] = (int)radix.size();
            nfac_of_q[q] = (int)g.size();
            for (int v : g) radix.push_back(v);
            psh_of_q[q] = pad_shift(g, (n & (n - 1)) == 0);
        }
        int maxp = 1;
        for (int v : f) maxp = v > maxp ? v : maxp;
        int lc = 0;
        if (maxp >= BLUESTEIN_MIN_PRIME) {
            lc = bluestein_len(2 * n - 1);
            if (lc > RING_EMAX) lc = 0;                  // does not fit one CTA: stay with the direct stage
        }
        lc_of_q[q] = lc;
        if (lc) {
            if (!pow2_tw_off.count(lc)) {
                pow2_tw_off[lc] = (int)tw.size();
                for (int j = 0; j < 2 * lc; ++j) {
                    long double ang = PI_LD * (long double)j / (long double)lc;
                    tw.push_back(make_double2((double)cosl(ang), (double)-sinl(ang)));
                }
                std::vector<int> pf, pg;
                factorize_ring(lc, pf);                  // 4s, a 2, then at most one 3 or 5
                group_radices(pf, pg);
                pow2_fac_off[lc] = (int)radix.size();
                for (int v : pg) radix.push_back(v);
                pow2_nfac[lc] = (int)pg.size();
                pow2_psh[lc] = pad_shift(pg, (lc & (lc - 1)) == 0);
            }
            // filter h_j = conj(c_j) = exp(+i pi j^2 / n) at j = -(n-1) .. n-1 (mod lc); Hf = FFT_lc(h) / lc
            std::vector<long double> hr(lc, 0.0L), hi(lc, 0.0L);
            for (int j = 0; j < n; ++j) {
                const long long e = ((long long)j * j) % (2LL * n);
                const long double ang = PI_LD * (long double)e / (long double)n;
                hr[j] = cosl(ang); hi[j] = sinl(ang);
                if (j > 0) { hr[lc - j] = hr[j]; hi[lc - j] = hi[j]; }
            }
            host_fft(hr, hi);
            hf_off_of_q[q] = (int)tw.size();
            std::vector<int> lf;
            factorize_ring(lc, lf);
            std::vector<double2> hf(lc);
            for (int k = 0; k < lc; ++k) {
                int kk = k, pos = 0, M = lc;
                for (int v : lf) { const int sdig = kk % v; kk /= v; M /= v; pos += sdig * M; }
                hf[pos] = make_double2((double)(hr[k] / lc), (double)(hi[k] / lc));
            }
            tw.insert(tw.end(), hf.begin(), hf.end());
            // chirp c_j = W_{2n}^{j^2 mod 2n}, j < n, right behind Hf (the kernels index it by j: no modulo per element)
            for (int j = 0; j < n; ++j) {
                const double2 cj = tw[tw_off_of_q[q] + (int)(((long long)j * j) % (2LL * n))];
                tw.push_back(cj);
            }
        }
        // forward (decimation in frequency) output order: bin k = s_1 + R_1 (s_2 + R_2 (...)) sits at
        // position s_1 n/R_1 + s_2 n/(R_1 R_2) + ...
        perm_off_of_q[q] = (int)perm.size();
        for (int k = 0; k < n; ++k) {
            int kk = k, pos = 0, M = n;
            for (int v : f) { const int sdig = kk % v; kk /= v; M /= v; pos += sdig * M; }
            perm.push_back((unsigned short)pos);
        }
    }
    // ---- mixed-radix fast path of the cap rings: N = 4 q = r1 r2 r3 with r1 >= r2 >= r3 >= 2 from the codelet set of
    // sht_ring_mixed.cu -- radices up to 16 if such a split exists (two CTAs per SM), else also 17, 19, 20, 23, 29, 31;
    // among the splits the one with the smallest largest radix (registers), then the largest smallest radix
    std::vector<int> mr1_of_q(nside + 1, 0), mr2_of_q(nside + 1, 0), mr3_of_q(nside + 1, 0);
    {
        const int small_set[] = {2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16};
        const int big_set[] = {2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 17, 19, 20, 23, 29, 31};
        for (int q = 1; q < nside; ++q) {
            const int n = 4 * q;
            if (n < MR_MIN_N || n > MR_MAX_N) continue;
            for (int pass = 0; pass < 2 && !mr1_of_q[q]; ++pass) {
                const int* set = pass == 0 ? small_set : big_set;
                const int ns_ = pass == 0 ? 15 : 21;
                int best[3] = {0, 0, 0};
                for (int ia = 0; ia < ns_; ++ia) {
                    const int a = set[ia];
                    if (n % a) continue;
                    for (int ib = 0; ib <= ia; ++ib) {
                        const int b = set[ib];
                        if ((n / a) % b) continue;
                        const int c = n / a / b;
                        if (c < 2 || c > b) continue;
                        bool ok = false;
                        for (int ic = 0; ic < ns_; ++ic) ok = ok || set[ic] == c;
                        if (!ok) continue;
                        if (!best[0] || a < best[0] || (a == best[0] && c > best[2])) { best[0] = a; best[1] = b; best[2] = c; }
                    }
                }
                if (best[0]) { mr1_of_q[q] = best[0]; mr2_of_q[q] = best[1]; mr3_of_q[q] = best[2]; }
            }
        }
    }
    // ---- chirp-z fast path of the cap rings: per ring length N = 4 q >= CZ_MIN_N with 2 N - 1 <= 4096 the filter spectrum
    // FFT_L(h) / L (h_j = exp(+i pi j^2 / N) at j = -(N-1) .. N-1 mod L; long double, natural order) and the chirp
    std::vector<int> cz_len_of_q(nside + 1, 0), cz_off_of_q(nside + 1, 0);
    int cz_tw_off[CZ_NCLASS];
    {
        std::vector<int> todo;
        for (int q = 1; q < nside; ++q) {
            const int n = 4 * q;
            if (n < CZ_MIN_N || mr1_of_q[q]) continue;       // the mixed-radix path comes first
            for (int c = 0; c < CZ_NCLASS; ++c)
                if (CZ_LEN[c] >= 2 * n - 1) { cz_len_of_q[q] = CZ_LEN[c]; break; }
            if (cz_len_of_q[q]) {
                cz_off_of_q[q] = (int)tw.size();
                tw.resize(tw.size() + (size_t)cz_len_of_q[q] + n);
                todo.push_back(q);
            }
        }
        auto work = [&](size_t first, size_t step) {
            for (size_t t = first; t < todo.size(); t += step) {
                const int q = todo[t], n = 4 * q, L = cz_len_of_q[q];
                std::vector<long double> hr(L, 0.0L), hi(L, 0.0L);
                for (int j = 0; j < n; ++j) {
                    const long long e = ((long long)j * j) % (2LL * n);
                    const long double ang = PI_LD * (long double)e / (long double)n;
                    hr[j] = cosl(ang); hi[j] = sinl(ang);
                    if (j > 0) { hr[L - j] = hr[j]; hi[L - j] = hi[j]; }
                }
                host_fft(hr, hi);
                double2* dst = tw.data() + cz_off_of_q[q];
                for (int k = 0; k < L; ++k) dst[k] = make_double2((double)(hr[k] / L), (double)(hi[k] / L));
                for (int j = 0; j < n; ++j) dst[L + j] = tw[tw_off_of_q[q] + (int)(((long long)j * j) % (2LL * n))];
            }
        };
        unsigned nthr = std::thread::hardware_concurrency();
        if (nthr < 1) nthr = 1;
        if (nthr > 16) nthr = 16;
        std::vector<std::thread> pool;
        for (unsigned t = 1; t < nthr; ++t) pool.emplace_back(work, (size_t)t, (size_t)nthr);
        work(0, nthr);
        for (auto& th : pool) th.join();
        for (int c = 0; c < CZ_NCLASS; ++c) {                // W_L^e, e < L
            cz_tw_off[c] = (int)tw.size();
            const int L = CZ_LEN[c];
            for (int e = 0; e < L; ++e) {
                const long double ang = 2.0L * PI_LD * (long double)e / (long double)L;
                tw.push_back(make_double2((double)cosl(ang), (double)-sinl(ang)));
            }
        }
    }
    const long long ns = nside;
    for (int p = 0; p < d.nh; ++p) {
        const long long i = p + 1;                       // north ring index, 1 .. 2 nside
        RingPair& r = rings[p];
        long double absz, s2;
        if (i < ns) {
            r.n = (int)(4 * i);
            long double omz = (long double)(i * i) / (long double)(3 * ns * ns);
            absz = 1.0L - omz; s2 = omz * (2.0L - omz);
            r.shift = 1;
            r.start_n = 2 * i * (i - 1);
        } else {
            r.n = (int)(4 * ns);
            absz = (long double)(4 * ns - 2 * i) / (long double)(3 * ns);
            s2 = (1.0L - absz) * (1.0L + absz);
            r.shift = ((i - ns) % 2 == 0) ? 1 : 0;
            r.start_n = 2 * ns * (ns - 1) + (i - ns) * 4 * ns;
        }
        r.start_s = (i == 2 * ns) ? -1 : d.npix - r.start_n - r.n;
        const int q = r.n / 4;
        r.tw_off = tw_off_of_q[q]; r.fac_off = fac_off_of_q[q]; r.nfac = nfac_of_q[q];
        r.perm_off = perm_off_of_q[q];
        r.lc = lc_of_q[q];
        r.b_tw_off = r.b_fac_off = r.b_nfac = r.hf_off = 0;
        if (r.lc) {
            r.b_tw_off = pow2_tw_off[r.lc]; r.b_fac_off = pow2_fac_off[r.lc]; r.b_nfac = pow2_nfac[r.lc];
            r.hf_off = hf_off_of_q[q];
            r.oop = 0;
            r.psh = pow2_psh[r.lc];
            r.nbuf = r.lc + (r.lc >> r.psh);
        } else {
            r.oop = nbig_of_q[q] >= 2 ? 1 : 0;
            r.psh = psh_of_q[q];
            r.nbuf = r.n + (r.n >> r.psh);
        }
        r.kt = ring_kt((size_t)r.nbuf * sizeof(double2) * (r.oop ? 2 : 1));
        r.pbits = 0; r.pm_hi = r.pm_lo = r.pm_keep = 0;
        if (!r.lc && (r.n & (r.n - 1)) == 0) {
            int a = 0;
            while ((1 << a) < r.n) ++a;
            // plain factor list of a power of two: 4s, then at most one 2; digit of width w at bits [lo, lo + w) of the bin
            int lo = 0;
            for (int rem = r.n; rem > 1;) {
                const int w = (rem % 4 == 0) ? 2 : 1;
                if (w == 2) { r.pm_hi |= 1u << (a - 1 - lo); r.pm_lo |= 1u << (a - 2 - lo); }
                else r.pm_keep |= 1u << (a - 1 - lo);
                lo += w; rem >>= w;
            }
            r.pbits = a;
        }
        r.mr_r1 = (i < ns) ? mr1_of_q[q] : 0; r.mr_r2 = mr2_of_q[q]; r.mr_r3 = mr3_of_q[q];
        r.cz_len = (i < ns) ? cz_len_of_q[q] : 0;
        r.cz_off = cz_off_of_q[q];
        r.mlim = lmax + 1;                               // tightened below from the l_safe table
        zs[p] = (double)absz; sin2s[p] = (double)s2;
    }

    // ---- recurrence coefficients (alpha_lm, beta_lm), m-major ---------------------------------
    //   lambda_l = alpha_l z lambda_{l-1} - beta_l lambda_{l-2},
    //   alpha_lm = sqrt((4 l^2 - 1)/(l^2 - m^2)),  beta_lm = alpha_lm / alpha_{l-1,m}
    //   slot l = m holds (0, -1) so that the same step reproduces the seed lambda_mm from the state (0, lambda_mm).
    std::vector<double2> coef((size_t)d.nalm);
    std::vector<double> cm(lmax + 1);
    {
        long double c = sqrtl(1.0L / (4.0L * PI_LD));
        cm[0] = (double)c;
        for (int m = 1; m <= lmax; ++m) { c = -c * sqrtl((2.0L * m + 1.0L) / (2.0L * m)); cm[m] = (double)c; }
    }
    for (int m = 0; m <= lmax; ++m) {
        const size_t base = (size_t)((long long)m * (2 * lmax + 1 - m) / 2);
        long double aprev = 0.0L;
        coef[base + m] = make_double2(0.0, -1.0);
        for (int l = m + 1; l <= lmax; ++l) {
            long double l2 = (long double)l * l, m2 = (long double)m * m;
            long double a = sqrtl((4.0L * l2 - 1.0L) / (l2 - m2));
            long double b = (l == m + 1) ? 0.0L : a / aprev;
            coef[base + l] = make_double2((double)a, (double)b);
            aprev = a;
        }
    }
    // spin-2 per-l constants: N_l = 2 / sqrt((l-1) l (l+1) (l+2)); (unused slots for l < 2 are 0)
    std::vector<double2> spin2c(lmax + 1, make_double2(0.0, 0.0));
    for (int l = 2; l <= lmax; ++l) {
        long double L = l;
        spin2c[l] = make_double2((double)(2.0L / sqrtl((L - 1.0L) * L * (L + 1.0L) * (L + 2.0L))), 0.0);
    }

    const double* d_cm = nullptr;
    if ((ce = upload(pl, zs, &d.z)) != cudaSuccess ||
        (ce = upload(pl, sin2s, &d.sin2)) != cudaSuccess || (ce = upload(pl, tw, &d.tw)) != cudaSuccess ||
        (ce = upload(pl, radix, &d.radix)) != cudaSuccess || (ce = upload(pl, perm, &d.perm)) != cudaSuccess || (ce = upload(pl, coef, &d.coef)) != cudaSuccess ||
        (ce = upload(pl, spin2c, &d.spin2c)) != cudaSuccess || (ce = upload(pl, cm, &d_cm)) != cudaSuccess) {
        sht_plan_destroy(pl);
        return SHT_ERR_ALLOC;
    }

    // ---- l_safe / seed table ------------------------------------------------------------------
    {
        const size_t cells = (size_t)(lmax + 1) * d.nh;
        int* ls = nullptr; double2* sd = nullptr;
        if (cudaMalloc(&ls, cells * sizeof(int)) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
        pl->dev_allocs[pl->n_allocs++] = ls;
        if (cudaMalloc(&sd, cells * sizeof(double2)) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
        pl->dev_allocs[pl->n_allocs++] = sd;
        pl->table_bytes += cells * (sizeof(int) + sizeof(double2));
        d.lstart = ls; d.seed = sd;
        ce = launch_seed_table(d, d_cm, ls, sd, 0);
        if (ce == cudaSuccess) ce = cudaDeviceSynchronize();
        if (ce != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_CUDA; }

        // recurrence state every LEG_CS-th l
        {
            std::vector<long long> csoff(lmax + 2, 0);
            for (int m = 0; m <= lmax; ++m) csoff[m + 1] = csoff[m] + (lmax - m) / LEG_CS + 1;
            if (upload(pl, csoff, &d.csoff) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            const size_t bytes = (size_t)csoff[lmax + 1] * d.nh * sizeof(double2);
            double2* cs = nullptr;
            if (cudaMalloc(&cs, bytes) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            pl->dev_allocs[pl->n_allocs++] = cs;
            pl->table_bytes += bytes;
            d.cseed = cs;
            ce = launch_chunk_seeds(d, cs, 0);
            if (ce == cudaSuccess) ce = cudaDeviceSynchronize();
            if (ce != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_CUDA; }
        }

        // ring optimisation (item 10): ring p takes part in order m only if lambda_lm(theta_p) reaches
        // the threshold for some l <= lmax, i.e. l_safe(m, p) <= lmax.  mlim[p] = 1 + the largest such m, made
        // monotone towards the equator; the ring kernels and the Legendre kernels both use exactly this bound,
        // so a workspace cell is read iff it was written.
        std::vector<int> hls(cells);
        if (cudaMemcpy(hls.data(), ls, cells * sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_CUDA; }
        std::vector<int> mlim(d.nh, 1);
        int run = 1;
        for (int p = 0; p < d.nh; ++p) {
            int mm = 0;
            for (int m = lmax; m > 0; --m)
                if (hls[(size_t)m * d.nh + p] <= lmax) { mm = m; break; }
            if (mm + 1 > run) run = mm + 1;
            mlim[p] = run;
            rings[p].mlim = run;
        }
        // Alg. 3, hybrid sweep (sht_api.cu): a ring pair of N pixels with mlim - 1 <= N / 2 holds no two orders that share a
        // bin (m'' = +-m mod N needs m + m'' >= N or |m - m''| >= N), so its orders never correct one another.  gs_pstar =
        // start of the alias-free tail of the ring pairs, rounded up to the synthesis kernel's blocks of 64 ring pairs
        {
            int ps = d.nh;
            for (int p = d.nh - 1; p >= 0; --p) {
                if (mlim[p] - 1 <= rings[p].n / 2) ps = p; else break;
            }
            ps = (ps + 63) / 64 * 64;
            if (ps > d.nh) ps = d.nh;
            pl->gs_pstar = ps;
            int mc = ps > 0 ? mlim[ps - 1] : 0;          // mlim is monotone: no ring pair below ps takes part in an order >= mc
            pl->gs_mcut = (mc + 1) & ~1;
            // two-phase variant for 2 nside <= lmax < 4 nside: on a belt ring pair (4 nside pixels, every order < 4 nside) an
            // order m shares its bin only with 4 nside - m, so the orders below 2 nside never meet one another there, nor
            // do the orders from 2 nside on.  Belt ring pairs from the first block of 64 that lies inside the belt.
            pl->gs2_pstar = 0; pl->gs2_msplit = 0;
            const int b0 = ((nside - 1) + 63) / 64 * 64;         // ring pair nside - 1 is the first belt ring
            if (spin == 0 && lmax >= 2 * nside && lmax < 4 * nside && b0 + 64 <= d.nh) { pl->gs2_pstar = b0; pl->gs2_msplit = 2 * nside; }
        }
        // first ring pair of every (m, l tile) of the Legendre analysis kernel: the smallest p >= the ring-pruning
        // bound whose recurrence has started before the end of the tile (no monotonicity of l_safe assumed)
        d.ntile_max = lmax / LEG_A_ML + 1;
        std::vector<int> pst((size_t)(lmax + 1) * d.ntile_max, d.nh);
        for (int m = 0; m <= lmax; ++m) {
            int* row = pst.data() + (size_t)m * d.ntile_max;
            const int nt = (lmax - m) / LEG_A_ML + 1;
            for (int p = 0; p < d.nh; ++p) {
                if (mlim[p] <= m) continue;
                const int lsv = hls[(size_t)m * d.nh + p];
                if (lsv > lmax) continue;
                const int jt = (lsv - m) / LEG_A_ML;
                if (jt < nt && p < row[jt]) row[jt] = p;
            }
            for (int t = 1; t < nt; ++t) if (row[t - 1] < row[t]) row[t] = row[t - 1];
        }
        if ((ce = upload(pl, pst, &d.pst)) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
        // block tables of the staged-lambda mode (the same loops as the contraction kernels)
        {
            d.npb = (d.nh + 63) / 64;
            std::vector<int> aoff((size_t)(lmax + 1) * d.ntile_max, 0), soff((size_t)(lmax + 1) * d.npb, 0),
                scf((size_t)(lmax + 1) * d.npb, lmax + 1), sm8((size_t)(lmax + 1) * d.npb * 8, lmax + 1);
            long long na = 0, nsb = 0;
            d.nck_max = 0; d.nst_max = 0;
            for (int m = 0; m <= lmax; ++m) {
                const int nt = (lmax - m) / LEG_A_ML + 1;
                for (int t = 0; t < nt; ++t) {
                    aoff[(size_t)m * d.ntile_max + t] = (int)na;
                    const int p0 = pst[(size_t)m * d.ntile_max + t];
                    const int apc = spin == 2 ? 16 : 32;               // rings per analysis stage
                    const int nck = p0 < d.nh ? (d.nh - p0 + apc - 1) / apc : 0;
                    na += nck;
                    if (nck > d.nck_max) d.nck_max = nck;
                }
                for (int b = 0; b < d.npb; ++b) {
                    soff[(size_t)m * d.npb + b] = (int)nsb;
                    const int plast = (b * 64 + 64 < d.nh ? b * 64 + 64 : d.nh) - 1;
                    if (m >= mlim[plast]) continue;
                    int lmin = lmax + 1;
                    for (int p = b * 64; p <= plast; ++p) {
                        const int lsv = hls[(size_t)m * d.nh + p];
                        lmin = lsv < lmin ? lsv : lmin;
                        int& q = sm8[((size_t)m * d.npb + b) * 8 + (p - b * 64) / 8];
                        q = lsv < q ? lsv : q;
                    }
                    if (lmin > lmax) continue;
                    const int cf = m + ((lmin - m) / 32) * 32;
                    scf[(size_t)m * d.npb + b] = cf;
                    const int nst = (lmax - cf) / 32 + 1;
                    nsb += nst;
                    if (nst > d.nst_max) d.nst_max = nst;
                }
            }
            // DMMA flops one k-tile (64 maps = 128 real columns) EXECUTES per direction (spin 0): the contraction
            // kernels' own skip logic (ring pruning per l tile, l_safe row blocks, blocks past lmax) replayed on the host
            // tables -- what bench.py divides by the time for the hardware-rate roofline fraction
            pl->exec_flops_tile[0] = pl->exec_flops_tile[1] = 0.0;
            if (spin == 0) {
                double fa = 0.0, fs = 0.0;
                for (int m = 0; m <= lmax; ++m) {
                    const int nt = (lmax - m) / LEG_A_ML + 1;
                    for (int t = 0; t < nt; ++t) {
                        const int l0 = m + t * LEG_A_ML;
                        const int i1 = std::min(8, (lmax - l0) / 16 + 1);
                        for (int pc = pst[(size_t)m * d.ntile_max + t]; pc < d.nh; pc += 32) {
                            int v[4]; bool plain = true;
                            for (int g = 0; g < 4; ++g) {
                                int lsmin = lmax + 1;
                                for (int p = pc + 8 * g; p < pc + 8 * g + 8 && p < d.nh; ++p) lsmin = std::min(lsmin, hls[(size_t)m * d.nh + p]);
                                v[g] = std::max(0, std::min(8, (lsmin - l0) >> 4));
                                plain = plain && v[g] == 0;
                            }
                            long long units = 0;
                            if (plain) units = 4LL * (i1 > 6 ? 8 : i1 > 4 ? 6 : i1 > 2 ? 4 : 2);
                            else for (int g = 0; g < 4; ++g) units += std::max(0, i1 - v[g]);
                            fa += (double)units * (2.0 * 16 * 8 * 128);
                        }
                    }
                    for (int b = 0; b < d.npb; ++b) {
                        const int cf = scf[(size_t)m * d.npb + b];
                        const int plast = (b * 64 + 64 < d.nh ? b * 64 + 64 : d.nh) - 1;
                        if (m >= mlim[plast] || cf > lmax) continue;
                        const int* q = &sm8[((size_t)m * d.npb + b) * 8];
                        for (int lc = cf; lc <= lmax; lc += 32) {
                            const int ks1 = std::min(4, (lmax - lc) / 8 + 1);
                            long long units = 0;
                            for (int ks = 0; ks < ks1; ++ks)
                                for (int i = 0; i < 8; ++i) units += q[i] <= lc + 8 * ks + 7 ? 1 : 0;
                            bool all0 = true;
                            for (int i = 0; i < 8; ++i) all0 = all0 && q[i] <= lc + 7;
                            if (all0 && ks1 == 4) units = 32;
                            fs += (double)units * (2.0 * 8 * 8 * 128);
                        }
                    }
                }
                pl->exec_flops_tile[0] = fa; pl->exec_flops_tile[1] = fs;
            } else {
                // spin 2 (E and B together), per k-tile of 32 pairs = 128 real columns: the analysis kernel runs the first
                // NI 16-row blocks of every chunk of 16 ring pairs from the tile's first ring on, the synthesis kernel
                // every step of 4 + 4 l of its stages that reaches down to l <= lmax; both multiply by F+ and by F-
                double fa = 0.0, fs = 0.0;
                for (int m = 0; m <= lmax; ++m) {
                    const int nt = (lmax - m) / LEG_A_ML + 1;
                    for (int t = 0; t < nt; ++t) {
                        const int l0 = m + t * LEG_A_ML;
                        const int i1 = std::min(8, (lmax - l0) / 16 + 1);
                        const int ni = i1 > 6 ? 8 : i1 > 4 ? 6 : i1 > 2 ? 4 : 2;
                        const int p0 = pst[(size_t)m * d.ntile_max + t];
                        if (p0 < d.nh) fa += (double)((d.nh - p0 + 15) / 16) * ni * (2.0 * 16 * 16 * 128 * 2);
                    }
                    for (int b = 0; b < d.npb; ++b) {
                        const int cf = scf[(size_t)m * d.npb + b];
                        const int plast = (b * 64 + 64 < d.nh ? b * 64 + 64 : d.nh) - 1;
                        if (m >= mlim[plast] || cf > lmax) continue;
                        for (int lc = cf; lc <= lmax; lc += 32)
                            fs += (double)std::min(8, 2 * ((lmax - lc) / 8 + 1)) * (2.0 * 4 * 64 * 128 * 2);
                    }
                }
                pl->exec_flops_tile[0] = fa; pl->exec_flops_tile[1] = fs;
            }
            pl->n_ablk = na; pl->n_sblk = nsb;
            if (na > 0x7fffffffLL || nsb > 0x7fffffffLL) { sht_plan_destroy(pl); return SHT_ERR_UNSUPPORTED; }
            if (upload(pl, aoff, &d.ablk_off) != cudaSuccess || upload(pl, soff, &d.sblk_off) != cudaSuccess ||
                upload(pl, scf, &d.scfirst) != cudaSuccess || upload(pl, sm8, &d.sminls8) != cudaSuccess) {
                sht_plan_destroy(pl);
                return SHT_ERR_ALLOC;
            }
        }
        if ((ce = upload(pl, rings, &d.rings)) != cudaSuccess || (ce = upload(pl, mlim, &d.mlim)) != cudaSuccess) {
            sht_plan_destroy(pl);
            return SHT_ERR_ALLOC;
        }
    }

    // ---- ring-kernel launch classes (by dynamic shared memory per CTA) --------------------------
    {
        const size_t lim[RING_NCLASS] = {72 * 1024, 113 * 1024, 160 * 1024, 224 * 1024};
        std::vector<int> lists[RING_NCLASS];
        for (int c = 0; c < RING_NCLASS; ++c) { pl->class_smem[c] = 0; pl->class_ktmin[c] = 16; }
        for (int p = 0; p < d.nh; ++p) {
            const size_t b = (size_t)rings[p].nbuf * rings[p].kt * sizeof(double2) * (rings[p].oop ? 2 : 1);
            int c = 0;
            while (c < RING_NCLASS && b > lim[c]) ++c;
            if (c == RING_NCLASS) { sht_plan_destroy(pl); return SHT_ERR_UNSUPPORTED; }
            lists[c].push_back(p);
            if (b > pl->class_smem[c]) pl->class_smem[c] = b;
            if (rings[p].kt < pl->class_ktmin[c]) pl->class_ktmin[c] = rings[p].kt;
        }
        for (int c = 0; c < RING_NCLASS; ++c) {
            pl->class_count[c] = (int)lists[c].size();
            const int* dp = nullptr;
            if (upload(pl, lists[c], &dp) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            pl->class_rings[c] = const_cast<int*>(dp);
        }
        // belt fast path: nside a power of two with a ring length the compiled transforms cover
        pl->belt_logn = 0; pl->belt_first = nside - 1; pl->belt_count = nside + 1; pl->fast_ring = true;
        pl->leg_tsplit = LEG_TSPLIT_DEFAULT; pl->leg_nsplit = LEG_NSPLIT_DEFAULT;      // sht_plan_set_option changes them
        if ((nside & (nside - 1)) == 0 && 4 * nside >= 512 && 4 * nside <= 2048) {
            int a = 0;
            while ((1 << a) < 4 * nside) ++a;
            pl->belt_logn = a;
        }
        for (int c = 0; c < RING_NCLASS; ++c) {
            std::vector<int> nb;
            pl->class_ktmin_nb[c] = 16;
            for (int p : lists[c]) {
                if (pl->belt_logn && p >= pl->belt_first) continue;
                if (rings[p].cz_len || rings[p].mr_r1) continue;
                nb.push_back(p);
                if (rings[p].kt < pl->class_ktmin_nb[c]) pl->class_ktmin_nb[c] = rings[p].kt;
            }
            pl->class_count_nb[c] = (int)nb.size();
            const int* dp = nullptr;
            if (upload(pl, nb, &dp) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            pl->class_rings_nb[c] = const_cast<int*>(dp);
        }
        for (int c = 0; c < 2 * MR_NCLASS; ++c) {            // mixed-radix classes: length class + 3 (radix above 16)
            std::vector<int> lst;
            int nmax = 0;
            for (int p = d.nh - 1; p >= 0; --p) {
                const RingPair& r = rings[p];
                if (!r.mr_r1) continue;
                const int lc = r.n <= 512 ? 0 : r.n <= 1024 ? 1 : 2;
                const int big = (r.mr_r1 > 16) ? 1 : 0;
                if (lc + MR_NCLASS * big != c) continue;
                lst.push_back(p);
                if (r.n > nmax) nmax = r.n;
            }
            pl->mr_count[c] = (int)lst.size();
            pl->mr_nmax[c] = nmax;
            const int* dp = nullptr;
            if (upload(pl, lst, &dp) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            pl->mr_rings[c] = const_cast<int*>(dp);
        }
        for (int c = 0; c < CZ_NCLASS; ++c) {                // longest rings first
            std::vector<int> lst;
            for (int p = d.nh - 1; p >= 0; --p)
                if (rings[p].cz_len == CZ_LEN[c]) lst.push_back(p);
            pl->cz_count[c] = (int)lst.size();
            pl->cz_tw_off[c] = cz_tw_off[c];
            const int* dp = nullptr;
            if (upload(pl, lst, &dp) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
            pl->cz_rings[c] = const_cast<int*>(dp);
        }
    }

    // ---- workspace: T_m^k(theta) for one chunk of maps ----------------------------------------
    {
        size_t freeb = 0, totalb = 0;
        cudaMemGetInfo(&freeb, &totalb);
        const size_t per_map = (size_t)d.nh * (lmax + 1) * d.ncomp * 2 * sizeof(double2);
        size_t budget = (size_t)(0.6 * (double)freeb);
        const size_t cap = (size_t)64 << 30;
        if (budget > cap) budget = cap;
        if (workspace_limit && budget > workspace_limit) budget = workspace_limit;
        long long fit = (long long)(budget / per_map) / KTILE_MAPS * KTILE_MAPS;
        if (fit < KTILE_MAPS) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
        long long need = ((long long)nmaps + KTILE_MAPS - 1) / KTILE_MAPS * KTILE_MAPS;
        d.kpad = (int)(need < fit ? need : fit);
        d.nkg = d.kpad / KG;
        pl->chunk = d.kpad < nmaps ? d.kpad : nmaps;
        pl->F_bytes = per_map * d.kpad;
        if (cudaMalloc(&pl->F, pl->F_bytes) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_ALLOC; }
        // padded map columns are never written by the ring kernels: keep them finite (zero) forever
        if (cudaMemset(pl->F, 0, pl->F_bytes) != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_CUDA; }
    }
    // ---- staged-lambda scratch: default mode when it fits beside the workspace ------------------------
    pl->lam = nullptr; pl->lam_i0 = nullptr; pl->lam_mode = SHT_LAMBDA_FUSED; pl->lam_bytes = 0;
    {
        size_t freeb = 0, totalb = 0;
        cudaMemGetInfo(&freeb, &totalb);
        const size_t a = (size_t)pl->n_ablk * LAM_ABLK_BYTES, sb = (size_t)pl->n_sblk * LAM_SBLK_BYTES * (spin == 2 ? 2 : 1);
        const size_t need = (a > sb ? a : sb) + 1024;
        if (need <= ((size_t)40 << 30) && need <= freeb / 4) {
            if (cudaMalloc(&pl->lam, need) == cudaSuccess && cudaMalloc(&pl->lam_i0, ((size_t)pl->n_ablk + 1) * sizeof(int)) == cudaSuccess) {
                pl->lam_bytes = need;
                pl->lam_mode = SHT_LAMBDA_STAGED;
            } else {
                cudaGetLastError();
                if (pl->lam) { cudaFree(pl->lam); pl->lam = nullptr; }
            }
        }
    }
    if (cudaDeviceSynchronize() != cudaSuccess) { sht_plan_destroy(pl); return SHT_ERR_CUDA; }
    pl->err[0] = 0;
    *out = pl;
    return SHT_OK;
}

extern "C" sht_status_t sht_plan_destroy(sht_plan_t pl)
{
    if (!pl) return SHT_OK;
    cudaDeviceSynchronize();
    for (int i = 0; i < pl->n_allocs; ++i) cudaFree(pl->dev_allocs[i]);
    if (pl->F) cudaFree(pl->F);
    if (pl->Fmap) cudaFree(pl->Fmap);
    if (pl->upow) cudaFree(pl->upow);
    if (pl->lam) cudaFree(pl->lam);
    if (pl->lam_i0) cudaFree(pl->lam_i0);
    for (int i = 0; i < pl->cap_ev; ++i) {
        if (pl->ev0[i]) cudaEventDestroy(pl->ev0[i]);
        if (pl->ev1[i]) cudaEventDestroy(pl->ev1[i]);
    }
    free(pl->ev0); free(pl->ev1); free(pl->ev_stage);
    if (pl->hevent) cudaEventDestroy(pl->hevent);
    if (pl->cap_stream) cudaStreamDestroy(pl->cap_stream);
    for (int i = 0; i < 4; ++i) {
        if (pl->stage_maps[i]) cudaFree(pl->stage_maps[i]);
        if (pl->stage_alm[i]) cudaFree(pl->stage_alm[i]);
        if (pl->stage_maps_f32[i]) cudaFree(pl->stage_maps_f32[i]);
        if (pl->stage_alm_f32[i]) cudaFree(pl->stage_alm_f32[i]);
        if (pl->hstream[i]) cudaStreamDestroy(pl->hstream[i]);
    }
    free(pl);
    return SHT_OK;
}
