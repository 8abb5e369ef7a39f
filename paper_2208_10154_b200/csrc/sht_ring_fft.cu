// sht_ring_fft.cu -- subsystem (1): batched ring DFTs over the variable-length HEALPix rings with the phi0
// phase shift, the m -> FFT-bin mapping on the frequency circle, and the north/south fold.
//
//   analysis  (eq. 2 row 3, "FFT mapping"; App. A.1 :412-416):
//       T_m^k(theta_r) = dsigma e^{-i m phi0_r} G_r^k[m mod N_r],   G = forward DFT of the ring,
//       then E = T(north) + T(south), O = T(north) - T(south) for the ring pair (r, 4 nside - r).
//   synthesis (PAPER.md:66-70 eq. 4, :78): ring spectrum Y[b] = sum_{m = b mod N} (w_m/2) d_m
//       + sum_{m = -b mod N} (w_m/2) conj(d_m), d_m = e^{+i m phi0} T_m, followed by the backward DFT.
//
// One CTA owns one ring pair and `kt` maps.  The north and the south ring of a map are packed as the real
// and imaginary part of ONE complex sequence (two real transforms for the price of one complex transform);
// the complex FFT is an out-of-place Stockham autosort FFT in shared memory with a per-ring-length radix
// list (4, 2, then the odd primes of N/4; a generic radix-R pass covers every prime).  No cuFFT.
//
// Workspace layout (both directions): F[p][m][comp][h][k][2] doubles, h = 0/1 = E/O (analysis) or
// north/south (synthesis), k fastest so that the Legendre stage reads dense [ring x (re,im of 64 maps)] rows.
#include "sht_internal.h"

namespace sht {

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

// W_N^e = exp(-2 pi i e / N) from the W_{2N} table (exp(+...) if INV)
template <bool INV>
__device__ __forceinline__ double2 twiddle(const double2* __restrict__ tw2, int e)
{
    double2 w = __ldg(tw2 + 2 * e);
    if (INV) w.y = -w.y;
    return w;
}

// One Stockham pass of radix R over `in` (length N) into `out`; p = product of the radices already done.
template <bool INV>
__device__ void pass_radix4(const double2* in, double2* out, int N, int p, const double2* tw2, int tid, int nt)
{
    const int T = N >> 2, unit = N / (4 * p);
    for (int i = tid; i < T; i += nt) {
        const int k = i % p, e = k * unit;
        double2 u0 = in[i];
        double2 u1 = cmul(in[i + T], twiddle<INV>(tw2, e));
        double2 u2 = cmul(in[i + 2 * T], twiddle<INV>(tw2, 2 * e));
        double2 u3 = cmul(in[i + 3 * T], twiddle<INV>(tw2, 3 * e));
        double2 v0 = cadd(u0, u2), v1 = csub(u0, u2), v2 = cadd(u1, u3), d = csub(u1, u3);
        double2 v3 = INV ? make_double2(-d.y, d.x) : make_double2(d.y, -d.x);   // (+-i) (u1 - u3)
        const int j = (i - k) * 4 + k;
        out[j] = cadd(v0, v2);
        out[j + p] = cadd(v1, v3);
        out[j + 2 * p] = csub(v0, v2);
        out[j + 3 * p] = csub(v1, v3);
    }
}

template <bool INV>
__device__ void pass_radix2(const double2* in, double2* out, int N, int p, const double2* tw2, int tid, int nt)
{
    const int T = N >> 1, unit = N / (2 * p);
    for (int i = tid; i < T; i += nt) {
        const int k = i % p;
        double2 u0 = in[i];
        double2 u1 = cmul(in[i + T], twiddle<INV>(tw2, k * unit));
        const int j = (i - k) * 2 + k;
        out[j] = cadd(u0, u1);
        out[j + p] = csub(u0, u1);
    }
}

// generic radix: one thread per output element, R complex multiply-adds each
template <bool INV>
__device__ void pass_generic(const double2* in, double2* out, int N, int R, int p, const double2* tw2, int tid, int nt)
{
    const int T = N / R, pr = p * R, unit = N / pr, sstep = N / R;
    for (int o = tid; o < N; o += nt) {
        const int blk = o / pr, rem = o - blk * pr;
        const int s = rem / p, k = rem - s * p;
        const int i = blk * p + k;
        int es = (int)(((long long)k * unit + (long long)s * sstep) % N);
        int e = 0;
        double2 acc = make_double2(0.0, 0.0);
        for (int r = 0; r < R; ++r) {
            double2 w = twiddle<INV>(tw2, e);
            double2 v = in[i + r * T];
            acc.x = fma(v.x, w.x, fma(-v.y, w.y, acc.x));
            acc.y = fma(v.x, w.y, fma(v.y, w.x, acc.y));
            e += es; if (e >= N) e -= N;
        }
        out[o] = acc;
    }
}

// complex FFT of buf (length N) by all threads of the CTA; result is left in buf.
template <bool INV>
__device__ void fft_cta(double2* buf, double2* scratch, int N, const int* __restrict__ radix, int nfac,
                        const double2* __restrict__ tw2)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    double2* src = buf; double2* dst = scratch;
    int p = 1;
    for (int f = 0; f < nfac; ++f) {
        const int R = radix[f];
        if (R == 4) pass_radix4<INV>(src, dst, N, p, tw2, tid, nt);
        else if (R == 2) pass_radix2<INV>(src, dst, N, p, tw2, tid, nt);
        else pass_generic<INV>(src, dst, N, R, p, tw2, tid, nt);
        p *= R;
        __syncthreads();
        double2* t = src; src = dst; dst = t;
    }
    if (src != buf) {
        for (int i = tid; i < N; i += nt) buf[i] = src[i];
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// analysis: maps -> F (E/O folded, phase shifted, aliased to every m)
// grid (kblocks, nh, ncomp)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_ring_analysis(DevicePlan d, const double* __restrict__ maps,
                                                      double* __restrict__ F, int k0, int kmaps)
{
    extern __shared__ double2 smem[];
    const int p = blockIdx.y, comp = blockIdx.z;
    const RingPair rp = d.rings[p];
    const int N = rp.n, kt = rp.kt;
    const int kbase = blockIdx.x * kt;
    if (kbase >= kmaps) return;
    const int tid = threadIdx.x, nt = blockDim.x;
    double2* scratch = smem + (size_t)kt * N;
    const double2* tw2 = d.tw + rp.tw_off;
    const int* radix = d.radix + rp.fac_off;

    // load: z[n] = T_north[n] + i T_south[n]
    for (int kk = 0; kk < kt; ++kk) {
        double2* buf = smem + (size_t)kk * N;
        const int k = kbase + kk;
        if (k < kmaps) {
            const double* mp = maps + ((size_t)(k0 + k) * d.ncomp + comp) * d.npix;
            const double* north = mp + rp.start_n;
            const double* south = rp.start_s >= 0 ? mp + rp.start_s : nullptr;
            for (int n = tid; n < N; n += nt)
                buf[n] = make_double2(__ldg(north + n), south ? __ldg(south + n) : 0.0);
        } else {
            for (int n = tid; n < N; n += nt) buf[n] = make_double2(0.0, 0.0);
        }
    }
    __syncthreads();
    for (int kk = 0; kk < kt; ++kk) fft_cta<false>(smem + (size_t)kk * N, scratch, N, radix, rp.nfac, tw2);

    // FFT mapping: m -> bin on the frequency circle, phase, fold; k fastest in the output
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    const int total = (d.lmax + 1) * kt;
    const bool equator = rp.start_s < 0;
    for (int idx = tid; idx < total; idx += nt) {
        const int kk = idx % kt, m = idx / kt;
        if (kbase + kk >= kmaps) continue;
        const double2* Z = smem + (size_t)kk * N;
        const int b = m % N, bc = b == 0 ? 0 : N - b;
        const double2 A = Z[b], B = Z[bc];
        // G_north = (A + conj B)/2, G_south = (A - conj B)/(2i)
        const double2 gn = make_double2(0.5 * (A.x + B.x), 0.5 * (A.y - B.y));
        const double2 gs = make_double2(0.5 * (A.y + B.y), -0.5 * (A.x - B.x));
        double2 ph = __ldg(tw2 + (int)(((long long)m * rp.shift) % (2 * N)));     // e^{-i m phi0}
        ph.x *= dsig; ph.y *= dsig;
        double2 E, O;
        if (equator) { E = cmul(ph, gn); O = make_double2(0.0, 0.0); }
        else { E = cmul(ph, cadd(gn, gs)); O = cmul(ph, csub(gn, gs)); }
        const size_t row = (((size_t)p * (d.lmax + 1) + m) * d.ncomp + comp) * 2;
        double2* Fe = reinterpret_cast<double2*>(F) + row * d.kpad + kbase + kk;
        Fe[0] = E;
        Fe[d.kpad] = O;
    }
}

// ------------------------------------------------------------------------------------------------
// synthesis: F (north/south T_m) -> maps.  If sub_from != nullptr: maps = sub_from - synthesis.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_ring_synthesis(DevicePlan d, const double* __restrict__ F,
                                                       double* __restrict__ maps, int k0, int kmaps,
                                                       const double* __restrict__ sub_from, int ksub0)
{
    extern __shared__ double2 smem[];
    const int p = blockIdx.y, comp = blockIdx.z;
    const RingPair rp = d.rings[p];
    const int N = rp.n, kt = rp.kt;
    const int kbase = blockIdx.x * kt;
    if (kbase >= kmaps) return;
    const int tid = threadIdx.x, nt = blockDim.x;
    double2* scratch = smem + (size_t)kt * N;
    const double2* tw2 = d.tw + rp.tw_off;
    const int* radix = d.radix + rp.fac_off;
    const bool equator = rp.start_s < 0;

    // ring spectrum of the packed sequence: Zin[b] = Y_north[b] + i Y_south[b]
    const int total = N * kt;
    for (int idx = tid; idx < total; idx += nt) {
        const int kk = idx % kt, b = idx / kt;
        double2 yn = make_double2(0.0, 0.0), ys = make_double2(0.0, 0.0);
        if (kbase + kk < kmaps) {
            // m = b (mod N): + (w/2) d_m ;  m = -b (mod N): + (w/2) conj(d_m)
            for (int pass = 0; pass < 2; ++pass) {
                const int mfirst = pass == 0 ? b : (b == 0 ? 0 : N - b);
                for (int m = mfirst; m <= d.lmax; m += N) {
                    const double w = (m == 0) ? 0.5 : 1.0;
                    double2 ph = __ldg(tw2 + (int)(((long long)m * rp.shift) % (2 * N)));
                    ph.y = -ph.y;                                                   // e^{+i m phi0}
                    const size_t row = (((size_t)p * (d.lmax + 1) + m) * d.ncomp + comp) * 2;
                    const double2* Fr = reinterpret_cast<const double2*>(F) + row * d.kpad + kbase + kk;
                    double2 dn = cmul(ph, Fr[0]);
                    double2 ds = cmul(ph, Fr[d.kpad]);
                    if (pass == 1) { dn.y = -dn.y; ds.y = -ds.y; }
                    yn.x = fma(w, dn.x, yn.x); yn.y = fma(w, dn.y, yn.y);
                    ys.x = fma(w, ds.x, ys.x); ys.y = fma(w, ds.y, ys.y);
                }
            }
        }
        // Y_n + i Y_s
        smem[(size_t)kk * N + b] = equator ? yn : make_double2(yn.x - ys.y, yn.y + ys.x);
    }
    __syncthreads();
    for (int kk = 0; kk < kt; ++kk) fft_cta<true>(smem + (size_t)kk * N, scratch, N, radix, rp.nfac, tw2);

    for (int kk = 0; kk < kt; ++kk) {
        const int k = kbase + kk;
        if (k >= kmaps) break;
        const double2* buf = smem + (size_t)kk * N;
        const size_t off = ((size_t)(k0 + k) * d.ncomp + comp) * d.npix;
        double* north = maps + off + rp.start_n;
        double* south = equator ? nullptr : maps + off + rp.start_s;
        if (sub_from) {
            const size_t soff = ((size_t)(ksub0 + k) * d.ncomp + comp) * d.npix;
            const double* rn = sub_from + soff + rp.start_n;
            const double* rs = equator ? nullptr : sub_from + soff + rp.start_s;
            for (int n = tid; n < N; n += nt) {
                const double2 v = buf[n];
                north[n] = rn[n] - v.x;
                if (south) south[n] = rs[n] - v.y;
            }
        } else {
            for (int n = tid; n < N; n += nt) {
                const double2 v = buf[n];
                north[n] = v.x;
                if (south) south[n] = v.y;
            }
        }
    }
}

static int ring_kt_min(const sht_plan_s* pl)
{
    // the longest ring has the fewest maps per CTA; it decides the grid width (CTAs beyond a ring's own
    // count exit at once)
    return pl->ring_kt_min;
}

cudaError_t launch_ring_analysis(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_ring_analysis, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int ktmin = ring_kt_min(pl);
    dim3 grid((kmaps + ktmin - 1) / ktmin, d.nh, d.ncomp);
    k_ring_analysis<<<grid, 256, pl->fft_smem, st>>>(d, maps, F, k0, kmaps);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_ring_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps,
                                  const double* sub_from, int ksub0, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_ring_synthesis, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int ktmin = ring_kt_min(pl);
    dim3 grid((kmaps + ktmin - 1) / ktmin, d.nh, d.ncomp);
    k_ring_synthesis<<<grid, 256, pl->fft_smem, st>>>(d, F, maps, k0, kmaps, sub_from, ksub0);
    pl->launches++;
    return cudaGetLastError();
}

}  // namespace sht
