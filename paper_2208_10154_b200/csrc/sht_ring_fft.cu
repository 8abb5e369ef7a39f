// sht_ring_fft.cu -- subsystem (1): batched ring DFTs over the variable-length HEALPix rings with the phi0
// phase shift, the m -> FFT-bin mapping on the frequency circle, and the north/south fold.
//
//   analysis  (eq. 2 row 3, "FFT mapping"; App. A.1 :412-416):
//       T_m^k(theta_r) = dsigma e^{-i m phi0_r} G_r^k[m mod N_r],   G = forward DFT of the ring,
//       then E = T(north) + T(south), O = T(north) - T(south) for the ring pair (r, 4 nside - r).
//   synthesis (PAPER.md:66-70 eq. 4, :78): ring spectrum Y[b] = sum_{m = b mod N} (w_m/2) d_m
//       + sum_{m = -b mod N} (w_m/2) conj(d_m), d_m = e^{+i m phi0} T_m, followed by the backward DFT.
//
// One CTA owns one ring pair and `kt` maps (kt * N <= RING_EMAX complex elements, all resident in shared
// memory, map index fastest so that every pass touches shared memory contiguously).  The north and the south
// ring of a map are packed as the real and imaginary part of ONE complex sequence (two real transforms for
// the price of one complex transform).  The complex FFT is an in-place mixed-radix transform: forward =
// decimation in frequency (natural order in, digit-reversed out), backward = decimation in time (digit-
// reversed in, natural out), so no pass needs a second buffer and the bin <-> position permutation is folded
// into the FFT-mapping step through a plan-time table.  Radices 4, 2, 3, 5, 7 are register butterflies; a
// prime factor >= 11 of the ring length is a direct O(R^2) stage placed at the global-memory end of the
// transform (first forward stage / last backward stage, fused with the map load / store); a second such
// prime runs out of place between two shared buffers.  No cuFFT.
//
// Workspace layout (both directions): F[p][kg][m][comp][h][kk][2] doubles (sht_internal.h), h = 0/1 = E/O
// (analysis) or north/south (synthesis): a CTA writes / reads whole 128-byte lines for kt >= 4.
// Only m < mlim(p) is produced / consumed (ring optimisation).
// Spin 2: component 1 of the workspace holds i*U (PAPER.md:111, 215 item 1: "all-real" products).
#include "sht_internal.h"

namespace sht {

constexpr int NT = 2 * RING_THREADS;             // launch bound; CTAs run RING_THREADS threads (two per SM) or twice that

// Shared-memory position of element e of map kk: maps fastest, and for power-of-two transforms one element of padding
// every 2^psh elements, so that the last (stride 8 or 16) register pass is free of bank conflicts (psh = 31: none).
struct Lay {
    int ktsh, psh;
    __device__ __forceinline__ int operator()(int e, int kk) const { return ((e + (e >> psh)) << ktsh) + kk; }
};

// position of bin k in the forward-transformed buffer: computed for power-of-two rings, tabulated otherwise
struct BinPos {
    const unsigned short* perm;
    int pbits;
    unsigned hi, lo, keep;
    __device__ __forceinline__ int operator()(int k) const
    {
        if (pbits) {
            const unsigned r = __brev((unsigned)k) >> (32 - pbits);
            return (int)(((r & hi) >> 1) | ((r & lo) << 1) | (r & keep));
        }
        return (int)__ldg(perm + k);
    }
};

// exp(-2 pi i k / 16)
__host__ __device__ constexpr double w16_cos(int k)
{
    return (k & 15) == 0 ? 1.0 : (k & 15) == 1 ? 0.92387953251128675613 : (k & 15) == 2 ? 0.70710678118654752440
         : (k & 15) == 3 ? 0.38268343236508977173 : (k & 15) == 4 ? 0.0 : (k & 15) == 5 ? -0.38268343236508977173
         : (k & 15) == 6 ? -0.70710678118654752440 : (k & 15) == 7 ? -0.92387953251128675613 : (k & 15) == 8 ? -1.0
         : (k & 15) == 9 ? -0.92387953251128675613 : (k & 15) == 10 ? -0.70710678118654752440
         : (k & 15) == 11 ? -0.38268343236508977173 : (k & 15) == 12 ? 0.0 : (k & 15) == 13 ? 0.38268343236508977173
         : (k & 15) == 14 ? 0.70710678118654752440 : 0.92387953251128675613;
}
__host__ __device__ constexpr double w16_sin(int k) { return w16_cos(k + 4); }     // -sin(2 pi k/16) = cos(2 pi (k+4)/16)
// multiply by exp(-+ 2 pi i k / 16) (k compile-time), - forward, + if INV
template <int K, bool INV>
__device__ __forceinline__ double2 mul_w16(double2 a)
{
    constexpr int k = K & 15;
    if constexpr (k == 0) return a;
    else if constexpr (k == 4) return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    else if constexpr (k == 8) return make_double2(-a.x, -a.y);
    else if constexpr (k == 12) return INV ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
    else {
        constexpr double c = w16_cos(k), sn = INV ? -w16_sin(k) : w16_sin(k);      // w = c + i sn
        return make_double2(fma(a.x, c, -(a.y * sn)), fma(a.x, sn, a.y * c));
    }
}

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

// cos / sin of 2 pi k / R for the odd register radices
__host__ __device__ constexpr double dft_cos(int R, int k)
{
    return k == 0 ? 1.0
         : R == 3 ? -0.5
         : R == 5 ? ((k == 1 || k == 4) ? 0.3090169943749474241 : -0.8090169943749474241)
         : (k == 1 || k == 6) ? 0.62348980185873353053
         : (k == 2 || k == 5) ? -0.22252093395631440429
                              : -0.90096886790241912624;
}
__host__ __device__ constexpr double dft_sin(int R, int k)
{
    return k == 0 ? 0.0
         : R == 3 ? (k == 1 ? 0.86602540378443864676 : -0.86602540378443864676)
         : R == 5 ? (k == 1 ? 0.95105651629515357212 : k == 2 ? 0.58778525229247312917
                   : k == 3 ? -0.58778525229247312917 : -0.95105651629515357212)
         : (k == 1 ? 0.78183148246802980871 : k == 2 ? 0.97492791218182360702 : k == 3 ? 0.43388373911755812048
          : k == 4 ? -0.43388373911755812048 : k == 5 ? -0.97492791218182360702 : -0.78183148246802980871);
}

// R-point DFT in registers: u[s] <- sum_r u[r] exp(-+ 2 pi i r s / R)   (- forward, + if INV)
template <int R, bool INV>
__device__ __forceinline__ void bfly(double2 (&u)[R])
{
    if constexpr (R == 2) {
        const double2 a = u[0], b = u[1];
        u[0] = cadd(a, b); u[1] = csub(a, b);
    } else if constexpr (R == 4) {
        const double2 v0 = cadd(u[0], u[2]), v1 = csub(u[0], u[2]), v2 = cadd(u[1], u[3]), dd = csub(u[1], u[3]);
        const double2 v3 = INV ? make_double2(-dd.y, dd.x) : make_double2(dd.y, -dd.x);   // (+-i)(u1 - u3)
        u[0] = cadd(v0, v2); u[1] = cadd(v1, v3); u[2] = csub(v0, v2); u[3] = csub(v1, v3);
    } else {
        constexpr int H = (R - 1) / 2;
        double2 a[H], b[H];
#pragma unroll
        for (int j = 1; j <= H; ++j) { a[j - 1] = cadd(u[j], u[R - j]); b[j - 1] = csub(u[j], u[R - j]); }
        const double2 u0 = u[0];
        double2 sum = u0;
#pragma unroll
        for (int j = 0; j < H; ++j) sum = cadd(sum, a[j]);
        u[0] = sum;
#pragma unroll
        for (int s = 1; s <= H; ++s) {
            double2 re = u0, im = make_double2(0.0, 0.0);
#pragma unroll
            for (int j = 1; j <= H; ++j) {
                const double c = dft_cos(R, (j * s) % R), sn = dft_sin(R, (j * s) % R);
                re.x = fma(c, a[j - 1].x, re.x); re.y = fma(c, a[j - 1].y, re.y);
                im.x = fma(sn, b[j - 1].x, im.x); im.y = fma(sn, b[j - 1].y, im.y);
            }
            // forward: X_s = re - i im, X_{R-s} = re + i im; backward: the other way round
            const double2 lo = make_double2(re.x + im.y, re.y - im.x), hi = make_double2(re.x - im.y, re.y + im.x);
            u[s] = INV ? hi : lo;
            u[R - s] = INV ? lo : hi;
        }
    }
}

// ---- forward stages (decimation in frequency, in place) ------------------------------------------------
// Stage with sub-length L and radix R, M = L / R: for each block base (multiple of L) and j < M the elements
// base + j + r M are replaced by W_L^{j s} sum_r x_r W_R^{r s}.  GIN: first stage (L = N), reads the maps.
template <int R, bool GIN, class LD>
__device__ __forceinline__ void dif_stage(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, LD ld)
{
    const int M = L / R, nw = (N / R) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[R];
#pragma unroll
        for (int r = 0; r < R; ++r) u[r] = GIN ? ld(e0 + r * M, kk) : buf[lay(e0 + r * M, kk)];
        bfly<R, false>(u);
        if (M > 1) {
#pragma unroll
            for (int s = 1; s < R; ++s) u[s] = cmul(u[s], twiddle<false>(tw2, j * s * tstep));
        }
#pragma unroll
        for (int s = 0; s < R; ++s) buf[lay(e0 + s * M, kk)] = u[s];
    }
    __syncthreads();
}

// Two consecutive radix-4 stages (sub-lengths L and L/4) on the 16 elements base + j + c L/16 held in registers:
// identical arithmetic and output order to dif_stage<4> twice, one shared-memory round trip instead of two.
template <bool GIN, class LD>
__device__ __forceinline__ void dif_stage16(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, LD ld)
{
    const int M = L >> 4, nw = (N >> 4) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) u[c] = GIN ? ld(e0 + c * M, kk) : buf[lay(e0 + c * M, kk)];
        double2 ta[4], tb[4];
        if (M > 1) {                                       // one table read; the other powers by multiplication
            ta[1] = twiddle<false>(tw2, j * tstep); ta[2] = cmul(ta[1], ta[1]); ta[3] = cmul(ta[1], ta[2]);
        }
        // stage A: radix 4 over the elements a + 4 r; twiddle W_L^{(j + a M) s} = W_L^{j s} W_16^{a s}
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            double2 v[4] = {u[a], u[a + 4], u[a + 8], u[a + 12]};
            bfly<4, false>(v);
            v[1] = a == 0 ? v[1] : a == 1 ? mul_w16<1, false>(v[1]) : a == 2 ? mul_w16<2, false>(v[1]) : mul_w16<3, false>(v[1]);
            v[2] = a == 0 ? v[2] : a == 1 ? mul_w16<2, false>(v[2]) : a == 2 ? mul_w16<4, false>(v[2]) : mul_w16<6, false>(v[2]);
            v[3] = a == 0 ? v[3] : a == 1 ? mul_w16<3, false>(v[3]) : a == 2 ? mul_w16<6, false>(v[3]) : mul_w16<9, false>(v[3]);
            if (M > 1) {
#pragma unroll
                for (int s = 1; s < 4; ++s) v[s] = cmul(v[s], ta[s]);
            }
#pragma unroll
            for (int s = 0; s < 4; ++s) u[a + 4 * s] = v[s];
        }
        // stage B: radix 4 inside each quarter s (elements 4 s + r'); twiddle W_{L/4}^{j s'}
        if (M > 1) { tb[1] = cmul(ta[2], ta[2]); tb[2] = cmul(tb[1], tb[1]); tb[3] = cmul(tb[1], tb[2]); }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            double2 v[4] = {u[4 * s], u[4 * s + 1], u[4 * s + 2], u[4 * s + 3]};
            bfly<4, false>(v);
            if (M > 1) {
#pragma unroll
                for (int q = 1; q < 4; ++q) v[q] = cmul(v[q], tb[q]);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) buf[lay(e0 + (4 * s + q) * M, kk)] = v[q];
        }
    }
    __syncthreads();
}

// A radix-4 stage (sub-length L) followed by a radix-2 stage (sub-length L/4) on 8 elements in registers.
template <bool GIN, class LD>
__device__ __forceinline__ void dif_stage8(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, LD ld)
{
    const int M = L >> 3, nw = (N >> 3) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) u[c] = GIN ? ld(e0 + c * M, kk) : buf[lay(e0 + c * M, kk)];
        double2 ta[4], tb;
        if (M > 1) {
            ta[1] = twiddle<false>(tw2, j * tstep); ta[2] = cmul(ta[1], ta[1]); ta[3] = cmul(ta[1], ta[2]);
            tb = cmul(ta[2], ta[2]);
        }
        // stage A: radix 4 over the elements a + 2 r; twiddle W_L^{(j + a M) s} = W_L^{j s} W_8^{a s}
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            double2 v[4] = {u[a], u[a + 2], u[a + 4], u[a + 6]};
            bfly<4, false>(v);
            if (a == 1) { v[1] = mul_w16<2, false>(v[1]); v[2] = mul_w16<4, false>(v[2]); v[3] = mul_w16<6, false>(v[3]); }
            if (M > 1) {
#pragma unroll
                for (int s = 1; s < 4; ++s) v[s] = cmul(v[s], ta[s]);
            }
#pragma unroll
            for (int s = 0; s < 4; ++s) u[a + 2 * s] = v[s];
        }
        // stage B: radix 2 inside each quarter s (elements 2 s, 2 s + 1); twiddle W_{L/4}^{j}
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const double2 x0 = cadd(u[2 * s], u[2 * s + 1]);
            double2 x1 = csub(u[2 * s], u[2 * s + 1]);
            if (M > 1) x1 = cmul(x1, tb);
            buf[lay(e0 + (2 * s) * M, kk)] = x0;
            buf[lay(e0 + (2 * s + 1) * M, kk)] = x1;
        }
    }
    __syncthreads();
}

// Direct stage for a prime 11 <= R <= 31: one thread owns a whole butterfly and keeps it in registers as the sums
// a_j = x_j + x_{R-j} and differences b_j = x_j - x_{R-j} (j = 1 .. H = (R-1)/2); the outputs s and R - s are then
// x_0 + sum_j cos(2 pi j s / R) a_j -+ i sum_j sin(2 pi j s / R) b_j: R^2 / 2 real multiply-adds per output pair, the
// cosines / sines read through the W_N table (the same address for the whole warp).  In place, no second buffer.
template <int R, bool GIN, class LD>
__device__ __forceinline__ void dif_prime(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, LD ld)
{
    constexpr int H = (R - 1) / 2;
    const int M = L / R, nw = (N / R) << lay.ktsh, tstep = N / L, rstep = 2 * (N / R);
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 a[H], b[H];
        const double2 x0 = GIN ? ld(e0, kk) : buf[lay(e0, kk)];
        double2 sum = x0;
#pragma unroll
        for (int q = 1; q <= H; ++q) {
            const double2 xa = GIN ? ld(e0 + q * M, kk) : buf[lay(e0 + q * M, kk)];
            const double2 xb = GIN ? ld(e0 + (R - q) * M, kk) : buf[lay(e0 + (R - q) * M, kk)];
            a[q - 1] = cadd(xa, xb); b[q - 1] = csub(xa, xb);
            sum = cadd(sum, a[q - 1]);
        }
        buf[lay(e0, kk)] = sum;
        for (int sx = 1; sx <= H; ++sx) {
            double2 re = x0, im = make_double2(0.0, 0.0);
            int idx = 0;
#pragma unroll
            for (int q = 0; q < H; ++q) {
                idx += sx; if (idx >= R) idx -= R;
                const double2 wv = __ldg(tw2 + idx * rstep);             // (cos, -sin) of 2 pi (q+1) s / R
                re.x = fma(wv.x, a[q].x, re.x); re.y = fma(wv.x, a[q].y, re.y);
                im.x = fma(-wv.y, b[q].x, im.x); im.y = fma(-wv.y, b[q].y, im.y);
            }
            double2 lo = make_double2(re.x + im.y, re.y - im.x), hi = make_double2(re.x - im.y, re.y + im.x);
            if (M > 1) {
                lo = cmul(lo, twiddle<false>(tw2, j * sx * tstep));
                hi = cmul(hi, twiddle<false>(tw2, j * (R - sx) * tstep));
            }
            buf[lay(e0 + sx * M, kk)] = lo;
            buf[lay(e0 + (R - sx) * M, kk)] = hi;
        }
    }
    __syncthreads();
}

// direct O(R^2) stage for a prime R >= 11: one thread per output element; src -> dst (different buffers, or
// src = the maps when GIN)
template <bool GIN, class LD>
__device__ __forceinline__ void dif_generic(const double2* src, double2* dst, int N, int L, int R, int kt, Lay lay,
                                            const double2* __restrict__ tw2, LD ld)
{
    const int M = L / R, nout = N << lay.ktsh, tstep = N / L, rstep = N / R;
    for (int o = threadIdx.x; o < nout; o += blockDim.x) {
        const int kk = o & (kt - 1), pos = o >> lay.ktsh;
        const int blk = pos / L, rem = pos - blk * L;
        const int s = rem / M, j = rem - s * M;
        const int e0 = blk * L + j;
        const int es = s * rstep;                          // exponent step of W_N per r: r s N / R
        int e = 0;
        double2 acc = make_double2(0.0, 0.0);
        for (int r = 0; r < R; ++r) {
            const double2 x = GIN ? ld(e0 + r * M, kk) : src[lay(e0 + r * M, kk)];
            const double2 w = twiddle<false>(tw2, e);
            acc.x = fma(x.x, w.x, fma(-x.y, w.y, acc.x));
            acc.y = fma(x.x, w.y, fma(x.y, w.x, acc.y));
            e += es; if (e >= N) e -= N;
        }
        if (M > 1) acc = cmul(acc, twiddle<false>(tw2, j * s * tstep));
        dst[lay(pos, kk)] = acc;
    }
    __syncthreads();
}

// ---- backward stages (decimation in time, in place): the exact adjoints of the forward stages ----------
template <int R, bool GOUT, class ST>
__device__ __forceinline__ void dit_stage(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, ST st)
{
    const int M = L / R, nw = (N / R) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[R];
#pragma unroll
        for (int s = 0; s < R; ++s) u[s] = buf[lay(e0 + s * M, kk)];
        if (M > 1) {
#pragma unroll
            for (int s = 1; s < R; ++s) u[s] = cmul(u[s], twiddle<true>(tw2, j * s * tstep));
        }
        bfly<R, true>(u);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (GOUT) st(e0 + r * M, kk, u[r]);
            else buf[lay(e0 + r * M, kk)] = u[r];
        }
    }
    if (!GOUT) __syncthreads();
}

// adjoint of dif_stage16: the radix-4 stage of sub-length L/4, then the one of sub-length L, in registers
template <bool GOUT, class ST>
__device__ __forceinline__ void dit_stage16(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, ST st)
{
    const int M = L >> 4, nw = (N >> 4) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) u[c] = buf[lay(e0 + c * M, kk)];
        double2 ta[4], tb[4];
        if (M > 1) {
            ta[1] = twiddle<true>(tw2, j * tstep); ta[2] = cmul(ta[1], ta[1]); ta[3] = cmul(ta[1], ta[2]);
            tb[1] = cmul(ta[2], ta[2]); tb[2] = cmul(tb[1], tb[1]); tb[3] = cmul(tb[1], tb[2]);
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            double2 v[4] = {u[4 * s], u[4 * s + 1], u[4 * s + 2], u[4 * s + 3]};
            if (M > 1) {
#pragma unroll
                for (int q = 1; q < 4; ++q) v[q] = cmul(v[q], tb[q]);
            }
            bfly<4, true>(v);
#pragma unroll
            for (int q = 0; q < 4; ++q) u[4 * s + q] = v[q];
        }
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            double2 v[4] = {u[a], u[a + 4], u[a + 8], u[a + 12]};
            if (M > 1) {
#pragma unroll
                for (int s = 1; s < 4; ++s) v[s] = cmul(v[s], ta[s]);
            }
            v[1] = a == 0 ? v[1] : a == 1 ? mul_w16<1, true>(v[1]) : a == 2 ? mul_w16<2, true>(v[1]) : mul_w16<3, true>(v[1]);
            v[2] = a == 0 ? v[2] : a == 1 ? mul_w16<2, true>(v[2]) : a == 2 ? mul_w16<4, true>(v[2]) : mul_w16<6, true>(v[2]);
            v[3] = a == 0 ? v[3] : a == 1 ? mul_w16<3, true>(v[3]) : a == 2 ? mul_w16<6, true>(v[3]) : mul_w16<9, true>(v[3]);
            bfly<4, true>(v);
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                if (GOUT) st(e0 + (a + 4 * r) * M, kk, v[r]);
                else buf[lay(e0 + (a + 4 * r) * M, kk)] = v[r];
            }
        }
    }
    if (!GOUT) __syncthreads();
}

// adjoint of dif_stage8
template <bool GOUT, class ST>
__device__ __forceinline__ void dit_stage8(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, ST st)
{
    const int M = L >> 3, nw = (N >> 3) << lay.ktsh, tstep = N / L;
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 u[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) u[c] = buf[lay(e0 + c * M, kk)];
        double2 ta[4], tb;
        if (M > 1) {
            ta[1] = twiddle<true>(tw2, j * tstep); ta[2] = cmul(ta[1], ta[1]); ta[3] = cmul(ta[1], ta[2]);
            tb = cmul(ta[2], ta[2]);
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const double2 x0 = u[2 * s];
            const double2 x1 = M > 1 ? cmul(u[2 * s + 1], tb) : u[2 * s + 1];
            u[2 * s] = cadd(x0, x1);
            u[2 * s + 1] = csub(x0, x1);
        }
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            double2 v[4] = {u[a], u[a + 2], u[a + 4], u[a + 6]};
            if (M > 1) {
#pragma unroll
                for (int s = 1; s < 4; ++s) v[s] = cmul(v[s], ta[s]);
            }
            if (a == 1) { v[1] = mul_w16<2, true>(v[1]); v[2] = mul_w16<4, true>(v[2]); v[3] = mul_w16<6, true>(v[3]); }
            bfly<4, true>(v);
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                if (GOUT) st(e0 + (a + 2 * r) * M, kk, v[r]);
                else buf[lay(e0 + (a + 2 * r) * M, kk)] = v[r];
            }
        }
    }
    if (!GOUT) __syncthreads();
}

// adjoint of dif_prime (plain form: all R inputs in registers, every output a dot product with a row of conj W_R; the
// sum / difference form costs more registers here because the inputs carry their twiddles)
template <int R, bool GOUT, class ST>
__device__ __forceinline__ void dit_prime(double2* buf, int N, int L, int kt, Lay lay, const double2* __restrict__ tw2, ST st)
{
    const int M = L / R, nw = (N / R) << lay.ktsh, tstep = N / L, rstep = 2 * (N / R);
    for (int w = threadIdx.x; w < nw; w += blockDim.x) {
        const int kk = w & (kt - 1), bf = w >> lay.ktsh;
        const int blk = bf / M, j = bf - blk * M;
        const int e0 = blk * L + j;
        double2 x[R];
#pragma unroll
        for (int sx = 0; sx < R; ++sx) x[sx] = buf[lay(e0 + sx * M, kk)];
        if (M > 1) {
#pragma unroll
            for (int sx = 1; sx < R; ++sx) x[sx] = cmul(x[sx], twiddle<true>(tw2, j * sx * tstep));
        }
        double2 sum = x[0];
#pragma unroll
        for (int sx = 1; sx < R; ++sx) sum = cadd(sum, x[sx]);
        if (GOUT) st(e0, kk, sum); else buf[lay(e0, kk)] = sum;
        for (int r = 1; r < R; ++r) {
            double2 acc = x[0];
            int idx = 0;
#pragma unroll
            for (int sx = 1; sx < R; ++sx) {
                idx += r; if (idx >= R) idx -= R;
                double2 wv = __ldg(tw2 + idx * rstep);                   // conj W_R^{r s}
                wv.y = -wv.y;
                acc.x = fma(x[sx].x, wv.x, fma(-x[sx].y, wv.y, acc.x));
                acc.y = fma(x[sx].x, wv.y, fma(x[sx].y, wv.x, acc.y));
            }
            if (GOUT) st(e0 + r * M, kk, acc); else buf[lay(e0 + r * M, kk)] = acc;
        }
    }
    if (!GOUT) __syncthreads();
}

template <bool GOUT, class ST>
__device__ __forceinline__ void dit_generic(const double2* src, double2* dst, int N, int L, int R, int kt, Lay lay,
                                            const double2* __restrict__ tw2, ST st)
{
    const int M = L / R, nout = N << lay.ktsh, tstep = N / L, rstep = N / R;
    for (int o = threadIdx.x; o < nout; o += blockDim.x) {
        const int kk = o & (kt - 1), pos = o >> lay.ktsh;
        const int blk = pos / L, rem = pos - blk * L;
        const int r = rem / M, j = rem - r * M;
        const int e0 = blk * L + j;
        int es = j * tstep + r * rstep;                    // exponent step per s: s (j N / L + r N / R)
        if (es >= N) es -= N;
        int e = 0;
        double2 acc = make_double2(0.0, 0.0);
        for (int s = 0; s < R; ++s) {
            const double2 x = src[lay(e0 + s * M, kk)];
            const double2 w = twiddle<true>(tw2, e);
            acc.x = fma(x.x, w.x, fma(-x.y, w.y, acc.x));
            acc.y = fma(x.x, w.y, fma(x.y, w.x, acc.y));
            e += es; if (e >= N) e -= N;
        }
        if (GOUT) st(pos, kk, acc);
        else dst[lay(pos, kk)] = acc;
    }
    if (!GOUT) __syncthreads();
}

// ---- transform drivers -----------------------------------------------------------------------------------
// The plan's radix list holds 2, 3, 4, 5, 7, primes >= 11, and the codes 16 (two radix-4 stages fused in registers)
// and 8 (a radix-4 and a radix-2 stage fused).
// forward transform of length N over the radix list (first stage reads through `ld`); returns the buffer that
// holds the result (bin k at position perm[k])
template <class LD>
__device__ __forceinline__ double2* fft_forward(double2* smem, int N, int nbuf, const int* __restrict__ radix, int nfac, int kt,
                                                Lay lay, const double2* __restrict__ tw2, LD ld)
{
    double2* cur = smem;
    int L = N;
    for (int f = 0; f < nfac; ++f) {
        const int R = radix[f];
        if (f == 0) {
            switch (R) {
                case 2: dif_stage<2, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 3: dif_stage<3, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 4: dif_stage<4, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 5: dif_stage<5, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 7: dif_stage<7, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 8: dif_stage8<true>(cur, N, L, kt, lay, tw2, ld); break;
                case 16: dif_stage16<true>(cur, N, L, kt, lay, tw2, ld); break;
                case 11: dif_prime<11, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 13: dif_prime<13, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 17: dif_prime<17, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 19: dif_prime<19, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 23: dif_prime<23, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 29: dif_prime<29, true>(cur, N, L, kt, lay, tw2, ld); break;
                case 31: dif_prime<31, true>(cur, N, L, kt, lay, tw2, ld); break;
                default: dif_generic<true>(nullptr, cur, N, L, R, kt, lay, tw2, ld); break;
            }
        } else {
            switch (R) {
                case 2: dif_stage<2, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 3: dif_stage<3, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 4: dif_stage<4, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 5: dif_stage<5, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 7: dif_stage<7, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 8: dif_stage8<false>(cur, N, L, kt, lay, tw2, ld); break;
                case 16: dif_stage16<false>(cur, N, L, kt, lay, tw2, ld); break;
                case 11: dif_prime<11, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 13: dif_prime<13, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 17: dif_prime<17, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 19: dif_prime<19, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 23: dif_prime<23, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 29: dif_prime<29, false>(cur, N, L, kt, lay, tw2, ld); break;
                case 31: dif_prime<31, false>(cur, N, L, kt, lay, tw2, ld); break;
                default: {
                    double2* other = (cur == smem) ? smem + nbuf : smem;
                    dif_generic<false>(cur, other, N, L, R, kt, lay, tw2, ld);
                    cur = other;
                } break;
            }
        }
        L /= R;
    }
    return cur;
}

// backward transform: `cur` holds bin k at position perm[k]; the last stage writes through `st`
template <class ST>
__device__ __forceinline__ void fft_backward(double2* smem, double2* cur, int N, int nbuf, const int* __restrict__ radix, int nfac,
                                             int kt, Lay lay, const double2* __restrict__ tw2, ST st)
{
    int L = 1;
    for (int f = nfac - 1; f >= 0; --f) {
        const int R = radix[f];
        L *= R;
        if (f == 0) {
            switch (R) {
                case 2: dit_stage<2, true>(cur, N, L, kt, lay, tw2, st); break;
                case 3: dit_stage<3, true>(cur, N, L, kt, lay, tw2, st); break;
                case 4: dit_stage<4, true>(cur, N, L, kt, lay, tw2, st); break;
                case 5: dit_stage<5, true>(cur, N, L, kt, lay, tw2, st); break;
                case 7: dit_stage<7, true>(cur, N, L, kt, lay, tw2, st); break;
                case 8: dit_stage8<true>(cur, N, L, kt, lay, tw2, st); break;
                case 16: dit_stage16<true>(cur, N, L, kt, lay, tw2, st); break;
                case 11: dit_prime<11, true>(cur, N, L, kt, lay, tw2, st); break;
                case 13: dit_prime<13, true>(cur, N, L, kt, lay, tw2, st); break;
                case 17: dit_prime<17, true>(cur, N, L, kt, lay, tw2, st); break;
                case 19: dit_prime<19, true>(cur, N, L, kt, lay, tw2, st); break;
                case 23: dit_prime<23, true>(cur, N, L, kt, lay, tw2, st); break;
                case 29: dit_prime<29, true>(cur, N, L, kt, lay, tw2, st); break;
                case 31: dit_prime<31, true>(cur, N, L, kt, lay, tw2, st); break;
                default: dit_generic<true>(cur, nullptr, N, L, R, kt, lay, tw2, st); break;
            }
        } else {
            switch (R) {
                case 2: dit_stage<2, false>(cur, N, L, kt, lay, tw2, st); break;
                case 3: dit_stage<3, false>(cur, N, L, kt, lay, tw2, st); break;
                case 4: dit_stage<4, false>(cur, N, L, kt, lay, tw2, st); break;
                case 5: dit_stage<5, false>(cur, N, L, kt, lay, tw2, st); break;
                case 7: dit_stage<7, false>(cur, N, L, kt, lay, tw2, st); break;
                case 8: dit_stage8<false>(cur, N, L, kt, lay, tw2, st); break;
                case 16: dit_stage16<false>(cur, N, L, kt, lay, tw2, st); break;
                case 11: dit_prime<11, false>(cur, N, L, kt, lay, tw2, st); break;
                case 13: dit_prime<13, false>(cur, N, L, kt, lay, tw2, st); break;
                case 17: dit_prime<17, false>(cur, N, L, kt, lay, tw2, st); break;
                case 19: dit_prime<19, false>(cur, N, L, kt, lay, tw2, st); break;
                case 23: dit_prime<23, false>(cur, N, L, kt, lay, tw2, st); break;
                case 29: dit_prime<29, false>(cur, N, L, kt, lay, tw2, st); break;
                case 31: dit_prime<31, false>(cur, N, L, kt, lay, tw2, st); break;
                default: {
                    double2* other = (cur == smem) ? smem + nbuf : smem;
                    dit_generic<false>(cur, other, N, L, R, kt, lay, tw2, st);
                    cur = other;
                } break;
            }
        }
    }
}

// Bluestein (chirp-z) circular convolution of length Lc = 2^a, 3 2^a or 5 2^a, in place in `buf`:
//   buf <- IFFT_Lc( FFT_Lc(x) . Hf ),  x delivered by `ld` (first forward stage), result handed to `st` by the
// last backward stage when GOUT, else left in buf in natural order.  Hf is stored in forward-output position order.
template <bool GIN, bool GOUT, bool CONJ, class LD, class ST>
__device__ __forceinline__ void bluestein_conv(double2* buf, int Lc, const int* __restrict__ radix, int nfac, int kt, Lay lay,
                                               const double2* __restrict__ btw, const double2* __restrict__ hf, LD ld, ST st)
{
    int L = Lc;
    for (int f = 0; f < nfac; ++f) {
        const int R = radix[f];
        if (GIN && f == 0) {
            if (R == 16) dif_stage16<true>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 8) dif_stage8<true>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 4) dif_stage<4, true>(buf, Lc, L, kt, lay, btw, ld);
            else dif_stage<2, true>(buf, Lc, L, kt, lay, btw, ld);
        } else {
            if (R == 16) dif_stage16<false>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 8) dif_stage8<false>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 4) dif_stage<4, false>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 3) dif_stage<3, false>(buf, Lc, L, kt, lay, btw, ld);
            else if (R == 5) dif_stage<5, false>(buf, Lc, L, kt, lay, btw, ld);
            else dif_stage<2, false>(buf, Lc, L, kt, lay, btw, ld);
        }
        L /= R;
    }
    const int tot = Lc << lay.ktsh;
    for (int i = threadIdx.x; i < tot; i += blockDim.x) {
        const int e = i >> lay.ktsh, kk = i & (kt - 1);
        double2 h = __ldg(hf + e);
        if (CONJ) h.y = -h.y;
        const int a = lay(e, kk);
        buf[a] = cmul(buf[a], h);
    }
    __syncthreads();
    L = 1;
    for (int f = nfac - 1; f >= 0; --f) {
        const int R = radix[f];
        L *= R;
        if (GOUT && f == 0) {
            if (R == 16) dit_stage16<true>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 8) dit_stage8<true>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 4) dit_stage<4, true>(buf, Lc, L, kt, lay, btw, st);
            else dit_stage<2, true>(buf, Lc, L, kt, lay, btw, st);
        } else {
            if (R == 16) dit_stage16<false>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 8) dit_stage8<false>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 4) dit_stage<4, false>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 3) dit_stage<3, false>(buf, Lc, L, kt, lay, btw, st);
            else if (R == 5) dit_stage<5, false>(buf, Lc, L, kt, lay, btw, st);
            else dit_stage<2, false>(buf, Lc, L, kt, lay, btw, st);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// analysis: maps -> F (E/O folded, phase shifted, aliased to every m < mlim)
// grid (map blocks, rings of the launch class, ncomp)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT, 1) k_ring_analysis(DevicePlan d, const int* __restrict__ ring_list,
                                                     const double* __restrict__ maps, double* __restrict__ F,
                                                     int k0, int kmaps, double* __restrict__ upow)
{
    extern __shared__ double2 smem[];
    const int p = ring_list[blockIdx.y], comp = blockIdx.z;
    const RingPair rp = d.rings[p];
    const int N = rp.n, kt = rp.kt, ktsh = __ffs(kt) - 1;
    const Lay lay{ktsh, rp.psh};
    const int nbuf = rp.nbuf << ktsh;                     // elements of one transform buffer (padding included)
    const int kbase = blockIdx.x * kt;
    if (kbase >= kmaps) return;
    const int tid = threadIdx.x, nt = blockDim.x;
    const double2* tw2 = d.tw + rp.tw_off;
    const BinPos perm{d.perm + rp.perm_off, rp.pbits, rp.pm_hi, rp.pm_lo, rp.pm_keep};
    const bool equator = rp.start_s < 0;
    const bool blue = rp.lc > 0;
    const double2* chirp = d.tw + rp.hf_off + rp.lc;      // c_j = exp(-i pi j^2 / N), j < N (Bluestein rings)

    // z[n] = T_north[n] + i T_south[n] of map kbase + kk
    const size_t map_stride = (size_t)d.ncomp * d.npix;
    const double* mbase = maps + ((size_t)(k0 + kbase) * d.ncomp + comp) * d.npix;
    const long long sn = rp.start_n, ss = rp.start_s;
    auto ld = [&](int e, int kk) -> double2 {
        if (kbase + kk >= kmaps) return make_double2(0.0, 0.0);
        const double* mp = mbase + (size_t)kk * map_stride;
        return make_double2(__ldg(mp + sn + e), equator ? 0.0 : __ldg(mp + ss + e));
    };

    double2* cur = smem;
    if (!blue) {
        cur = fft_forward(smem, N, nbuf, d.radix + rp.fac_off, rp.nfac, kt, lay, tw2, ld);
    } else {
        // X_b = c_b sum_n (x_n c_n) conj(c)_{b-n},  c_n = exp(-i pi n^2 / N) = W_{2N}^{n^2 mod 2N}
        auto ldc = [&](int e, int kk) -> double2 {
            if (e >= N) return make_double2(0.0, 0.0);
            return cmul(ld(e, kk), __ldg(chirp + e));
        };
        auto nost = [](int, int, double2) {};
        bluestein_conv<true, false, false>(smem, rp.lc, d.radix + rp.b_fac_off, rp.b_nfac, kt, lay, d.tw + rp.b_tw_off,
                                           d.tw + rp.hf_off, ldc, nost);
    }

    // FFT mapping: m -> bin on the frequency circle (stored at position perm[bin]), phase, fold.
    // A thread keeps its map (nt is a multiple of kt) and walks m with a fixed stride: m mod N, m mod 2N and the
    // workspace address advance incrementally (no division, no 64-bit multiply in the loop).
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    const int kk = tid & (kt - 1), k = kbase + kk;
    if (k >= kmaps) return;
    const int dm = nt >> ktsh, dmN = dm % N, dm2N = dm % (2 * N);
    int m = tid >> ktsh;
    int b = m % N, m2 = m % (2 * N);
    const size_t cstride = (size_t)d.ncomp * 2 * KG;                       // double2 per order m
    double2* Fp = reinterpret_cast<double2*>(F) + f_cell(d, p, k >> 2, 0, comp, 0) + (k & 3) + (size_t)m * cstride;
    const int mlim = rp.mlim;
    if (upow && mlim <= N / 2) {
        // Alg. 2 in T_m-space: power of the ring pair in the bins no stored order m < mlim reaches (b = mlim .. N/2); the
        // residual of those bins never changes, its power enters the per-round rms through this table [p][comp][map]
        double acc = 0.0;
        for (int bb = mlim + (tid >> ktsh); bb <= N / 2; bb += dm) {
            const int bc2 = N - bb;
            double2 A, B;
            if (!blue) {
                A = cur[lay(perm(bb), kk)]; B = cur[lay(perm(bc2), kk)];
            } else {
                A = cmul(cur[lay(bb, kk)], __ldg(chirp + bb));
                B = cmul(cur[lay(bc2, kk)], __ldg(chirp + bc2));
            }
            const double2 gn = make_double2(0.5 * (A.x + B.x), 0.5 * (A.y - B.y));
            const double2 gs = make_double2(0.5 * (A.y + B.y), -0.5 * (A.x - B.x));
            const double w = (2 * bb == N) ? 1.0 : 2.0;
            acc += w * (gn.x * gn.x + gn.y * gn.y + (equator ? 0.0 : gs.x * gs.x + gs.y * gs.y));
        }
        if (acc != 0.0) atomicAdd(upow + ((size_t)p * d.ncomp + comp) * d.kpad + k, acc);
    }
#pragma unroll 4
    for (; m < mlim; m += dm) {
        const int bc = b == 0 ? 0 : N - b;
        double2 A, B;
        if (!blue) {
            A = cur[lay(perm(b), kk)]; B = cur[lay(perm(bc), kk)];
        } else {
            A = cmul(cur[lay(b, kk)], __ldg(chirp + b));
            B = cmul(cur[lay(bc, kk)], __ldg(chirp + bc));
        }
        // G_north = (A + conj B)/2, G_south = (A - conj B)/(2i)
        const double2 gn = make_double2(0.5 * (A.x + B.x), 0.5 * (A.y - B.y));
        const double2 gs = make_double2(0.5 * (A.y + B.y), -0.5 * (A.x - B.x));
        double2 ph = make_double2(dsig, 0.0);
        if (rp.shift) {                                   // e^{-i m phi0}, phi0 = pi / N
            ph = __ldg(tw2 + m2);
            ph.x *= dsig; ph.y *= dsig;
        }
        double2 E, O;
        if (equator) { E = cmul(ph, gn); O = make_double2(0.0, 0.0); }
        else { E = cmul(ph, cadd(gn, gs)); O = cmul(ph, csub(gn, gs)); }
        if (comp == 1) { E = make_double2(-E.y, E.x); O = make_double2(-O.y, O.x); }      // i U
        Fp[0] = E;
        Fp[KG] = O;
        Fp += (size_t)dm * cstride;
        b += dmN; if (b >= N) b -= N;
        m2 += dm2N; if (m2 >= 2 * N) m2 -= 2 * N;
    }
}

// ------------------------------------------------------------------------------------------------
// synthesis: F (north/south T_m) -> maps.  If sub_from != nullptr: maps = sub_from - synthesis.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT, 1) k_ring_synthesis(DevicePlan d, const int* __restrict__ ring_list,
                                                      const double* __restrict__ F, double* __restrict__ maps,
                                                      int k0, int kmaps, const double* __restrict__ sub_from, int ksub0)
{
    extern __shared__ double2 smem[];
    const int p = ring_list[blockIdx.y], comp = blockIdx.z;
    const RingPair rp = d.rings[p];
    const int N = rp.n, kt = rp.kt, ktsh = __ffs(kt) - 1;
    const Lay lay{ktsh, rp.psh};
    const int nbuf = rp.nbuf << ktsh;                     // elements of one transform buffer (padding included)
    const int kbase = blockIdx.x * kt;
    if (kbase >= kmaps) return;
    const int tid = threadIdx.x, nt = blockDim.x;
    const double2* tw2 = d.tw + rp.tw_off;
    const BinPos perm{d.perm + rp.perm_off, rp.pbits, rp.pm_hi, rp.pm_lo, rp.pm_keep};
    const bool equator = rp.start_s < 0;
    const bool blue = rp.lc > 0;
    const double2* chirp = d.tw + rp.hf_off + rp.lc;      // c_j = exp(-i pi j^2 / N), j < N (Bluestein rings)
    const int mlim = rp.mlim;
    // the Legendre synthesis stores the even and the odd sum of a ring pair: north = even + odd, south = even - odd
    double2* cur = smem;

    // ring spectrum of the packed sequence, Z[b] = Y_north[b] + i Y_south[b]; bins b <= N/2 are assembled
    // from the workspace (each cell read once), bins N - b follow from the Hermitian symmetry of Y_n, Y_s
    // A thread keeps its map and walks the bins with a fixed stride; workspace addresses advance incrementally.
    {
        const int kk = tid & (kt - 1), k = kbase + kk;
        const int db = nt >> ktsh;
        const size_t cstride = (size_t)d.ncomp * 2 * KG;                   // double2 per order m
        const double2* Fb = reinterpret_cast<const double2*>(F) + f_cell(d, p, (k < kmaps ? k : kbase) >> 2, 0, comp, 0) + (k & 3);
        for (int b = tid >> ktsh; b <= N / 2; b += db) {
            double2 yn = make_double2(0.0, 0.0), ys = make_double2(0.0, 0.0);
            if (k < kmaps) {
                // m = b (mod N): + (w/2) d_m ;  m = -b (mod N): + (w/2) conj(d_m);  d_m = e^{+i m phi0} T_m
#pragma unroll
                for (int pass = 0; pass < 2; ++pass) {
                    const int mfirst = pass == 0 ? b : (b == 0 ? 0 : N - b);
                    int m2 = mfirst;                                       // m mod 2N
                    const double2* Fp = Fb + (size_t)mfirst * cstride;
                    for (int m = mfirst; m < mlim; m += N, Fp += (size_t)N * cstride) {
                        const double w = (m == 0) ? 0.5 : 1.0;
                        double2 ph = make_double2(1.0, 0.0);
                        if (rp.shift) { ph = __ldg(tw2 + m2); ph.y = -ph.y; }
                        double2 fn = Fp[0], fs = Fp[KG];
                        { const double2 e = fn, o = fs; fn = cadd(e, o); fs = csub(e, o); }       // stored as (even, odd) sums
                        if (comp == 1) { fn = make_double2(fn.y, -fn.x); fs = make_double2(fs.y, -fs.x); }   // U = -i (iU)
                        double2 dn = cmul(ph, fn), ds = cmul(ph, fs);
                        if (pass == 1) { dn.y = -dn.y; ds.y = -ds.y; }
                        yn.x = fma(w, dn.x, yn.x); yn.y = fma(w, dn.y, yn.y);
                        ys.x = fma(w, ds.x, ys.x); ys.y = fma(w, ds.y, ys.y);
                        m2 += N; if (m2 >= 2 * N) m2 -= 2 * N;
                    }
                }
            }
            if (equator) ys = make_double2(0.0, 0.0);
            if (b == 0 || 2 * b == N) { yn.y = 0.0; ys.y = 0.0; }
            const double2 zb = make_double2(yn.x - ys.y, yn.y + ys.x);
            const double2 zc = make_double2(yn.x + ys.y, ys.x - yn.y);           // Z[N - b]
            if (!blue) {
                cur[lay(perm(b), kk)] = zb;
                if (b > 0 && 2 * b < N) cur[lay(perm(N - b), kk)] = zc;
            } else {
                // x_n = conj(c)_n sum_b (Z_b conj(c)_b) c_{n-b}
                double2 c = __ldg(chirp + b); c.y = -c.y;
                cur[lay(b, kk)] = cmul(zb, c);
                if (b > 0 && 2 * b < N) {
                    const int bb = N - b;
                    double2 c2 = __ldg(chirp + bb); c2.y = -c2.y;
                    cur[lay(bb, kk)] = cmul(zc, c2);
                }
            }
        }
    }
    if (blue) {
        const int tot = rp.lc << ktsh;
        for (int i = (N << ktsh) + tid; i < tot; i += nt) cur[lay(i >> ktsh, i & (kt - 1))] = make_double2(0.0, 0.0);
    }
    __syncthreads();

    const size_t map_stride = (size_t)d.ncomp * d.npix;
    double* obase = maps + ((size_t)(k0 + kbase) * d.ncomp + comp) * d.npix;
    const double* sbase = sub_from ? sub_from + ((size_t)(ksub0 + kbase) * d.ncomp + comp) * d.npix : nullptr;
    const long long sn = rp.start_n, ss = rp.start_s;
    auto st = [&](int e, int kk, double2 v) {
        if (kbase + kk >= kmaps) return;
        double* mp = obase + (size_t)kk * map_stride;
        if (sbase) {
            const double* sp = sbase + (size_t)kk * map_stride;
            mp[sn + e] = sp[sn + e] - v.x;
            if (!equator) mp[ss + e] = sp[ss + e] - v.y;
        } else {
            mp[sn + e] = v.x;
            if (!equator) mp[ss + e] = v.y;
        }
    };

    if (!blue) {
        fft_backward(smem, cur, N, nbuf, d.radix + rp.fac_off, rp.nfac, kt, lay, tw2, st);
    } else {
        auto stc = [&](int e, int kk, double2 v) {
            if (e >= N) return;
            double2 c = __ldg(chirp + e); c.y = -c.y;
            st(e, kk, cmul(v, c));
        };
        auto nold = [](int, int) -> double2 { return make_double2(0.0, 0.0); };
        bluestein_conv<false, true, true>(smem, rp.lc, d.radix + rp.b_fac_off, rp.b_nfac, kt, lay, d.tw + rp.b_tw_off,
                                          d.tw + rp.hf_off, nold, stc);
    }
}

// ------------------------------------------------------------------------------------------------
// Alg. 2 kept between T_m and a_lm (item 8): the ring FFTs are lossless, so the
// residual map - synthesis(a) is formed on the ring spectra.  F holds the synthesised T_m (north / south) of one round,
// Fmap the folded T_m of the input maps.  Per ring pair: the synthesised ring spectrum Y[b] is assembled exactly as in
// k_ring_synthesis, re-expanded to every m < mlim on the frequency circle (FFT(ring)[b] = N Y[b]; the phases and d sigma
// of the analysis side) and subtracted; F is overwritten with the folded residual.  By Parseval the sum of squares of the
// residual pixels of the pair is (1/N) sum_b |R[b]|^2: bins b < mlim from the residual itself, the others from `upow`.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT, 1) k_ring_residual(DevicePlan d, const int* __restrict__ ring_list,
                                                     double* __restrict__ F, const double* __restrict__ Fmap,
                                                     const double* __restrict__ upow, double* __restrict__ acc_out,
                                                     int kmaps)
{
    extern __shared__ double2 smem[];
    const int p = ring_list[blockIdx.y], comp = blockIdx.z;
    const RingPair rp = d.rings[p];
    const int N = rp.n, kt = rp.kt, ktsh = __ffs(kt) - 1;
    const int kbase = blockIdx.x * kt;
    if (kbase >= kmaps) return;
    const int tid = threadIdx.x, nt = blockDim.x;
    const double2* tw2 = d.tw + rp.tw_off;
    const bool equator = rp.start_s < 0;
    const int mlim = rp.mlim, nb = N / 2 + 1;
    double2* Yn = smem;                                   // [b][kk]
    double2* Ys = smem + ((size_t)nb << ktsh);
    const int kk = tid & (kt - 1), k = kbase + kk;
    const int db = nt >> ktsh;
    const size_t cstride = (size_t)d.ncomp * 2 * KG;
    const size_t cell0 = f_cell(d, p, (k < kmaps ? k : kbase) >> 2, 0, comp, 0) + (k & 3);
    const double2* Fs = reinterpret_cast<const double2*>(F) + cell0;
    // ---- ring spectrum of the synthesised pair (same arithmetic as k_ring_synthesis)
    for (int b = tid >> ktsh; b < nb; b += db) {
        double2 yn = make_double2(0.0, 0.0), ys = make_double2(0.0, 0.0);
        if (k < kmaps) {
#pragma unroll
            for (int pass = 0; pass < 2; ++pass) {
                const int mfirst = pass == 0 ? b : (b == 0 ? 0 : N - b);
                int m2 = mfirst;
                const double2* Fp = Fs + (size_t)mfirst * cstride;
                for (int m = mfirst; m < mlim; m += N, Fp += (size_t)N * cstride) {
                    const double w = (m == 0) ? 0.5 : 1.0;
                    double2 ph = make_double2(1.0, 0.0);
                    if (rp.shift) { ph = __ldg(tw2 + m2); ph.y = -ph.y; }
                    double2 fn = Fp[0], fs = Fp[KG];
                    { const double2 e = fn, o = fs; fn = cadd(e, o); fs = csub(e, o); }       // stored as (even, odd) sums
                    if (comp == 1) { fn = make_double2(fn.y, -fn.x); fs = make_double2(fs.y, -fs.x); }
                    double2 dn = cmul(ph, fn), ds = cmul(ph, fs);
                    if (pass == 1) { dn.y = -dn.y; ds.y = -ds.y; }
                    yn.x = fma(w, dn.x, yn.x); yn.y = fma(w, dn.y, yn.y);
                    ys.x = fma(w, ds.x, ys.x); ys.y = fma(w, ds.y, ys.y);
                    m2 += N; if (m2 >= 2 * N) m2 -= 2 * N;
                }
            }
        }
        if (equator) ys = make_double2(0.0, 0.0);
        if (b == 0 || 2 * b == N) { yn.y = 0.0; ys.y = 0.0; }
        Yn[(b << ktsh) + kk] = yn;
        Ys[(b << ktsh) + kk] = ys;
    }
    __syncthreads();
    if (k >= kmaps) return;
    // ---- residual of every order m < mlim, folded; sum of squares of the covered bins
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    const double scale = dsig * (double)N;                // FFT(ring)[b] = N Y[b], times d sigma of the analysis side
    const double2* Fm = reinterpret_cast<const double2*>(Fmap) + cell0;
    double2* Fo = reinterpret_cast<double2*>(F) + cell0;
    const int dmN = db % N, dm2N = db % (2 * N);
    int m = tid >> ktsh;
    int b = m % N, m2 = m % (2 * N);
    double ssq = 0.0;
    for (; m < mlim; m += db) {
        const bool cj = 2 * b > N;
        const int bb = cj ? N - b : b;
        double2 tn = Yn[(bb << ktsh) + kk], ts = Ys[(bb << ktsh) + kk];
        if (cj) { tn.y = -tn.y; ts.y = -ts.y; }
        double2 ph = make_double2(scale, 0.0);
        if (rp.shift) { ph = __ldg(tw2 + m2); ph.x *= scale; ph.y *= scale; }
        double2 se, so;
        if (equator) { se = cmul(ph, tn); so = make_double2(0.0, 0.0); }
        else { se = cmul(ph, cadd(tn, ts)); so = cmul(ph, csub(tn, ts)); }
        if (comp == 1) { se = make_double2(-se.y, se.x); so = make_double2(-so.y, so.x); }
        const size_t off = (size_t)m * cstride;
        const double2 E = csub(Fm[off], se), O = csub(Fm[off + KG], so);
        Fo[off] = E;
        Fo[off + KG] = O;
        if (2 * m <= N) {                                 // m is its own bin: |R_north|^2 + |R_south|^2 (times d sigma^2)
            const double w = (m == 0 || 2 * m == N) ? 1.0 : 2.0;
            const double q = equator ? (E.x * E.x + E.y * E.y)
                                     : 0.5 * (E.x * E.x + E.y * E.y + O.x * O.x + O.y * O.y);
            ssq = fma(w, q, ssq);
        }
        b += dmN; if (b >= N) b -= N;
        m2 += dm2N; if (m2 >= 2 * N) m2 -= 2 * N;
    }
    double tot = ssq / (dsig * dsig);
    if ((tid >> ktsh) == 0) tot += upow[((size_t)p * d.ncomp + comp) * d.kpad + k];
    if (tot != 0.0) atomicAdd(acc_out + (size_t)k * d.ncomp + comp, tot / (double)N);
}

// ------------------------------------------------------------------------------------------------
// Alg. 3 ("update F from delta T_m"; reading G21): the residual R (folded T_m of map - synthesis(a),
// all orders) is kept up to date order by order.  S holds, at order m only, the synthesised T_m (north / south) of the
// increment delta a_m; its ring spectrum has one bin, bb = the bin m falls on, and every order m'' < mlim of the ring
// pair that falls on the same bin (directly or as the conjugate) is corrected -- the arithmetic of k_ring_residual
// restricted to one source order.  One thread per (ring pair, map).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void gs_update_cell(const DevicePlan& d, const double* __restrict__ S, double* __restrict__ R, int p, int comp,
                                               int m, int k, int kmaps)
{
    const RingPair& rp = d.rings[p];
    const int N = rp.n, mlim = rp.mlim;
    if (k >= kmaps || m >= mlim) return;
    const double2* tw2 = d.tw + rp.tw_off;
    const bool equator = rp.start_s < 0, shift = rp.shift != 0;
    const size_t cstride = (size_t)d.ncomp * 2 * KG;
    const size_t cell0 = f_cell(d, p, k >> 2, 0, comp, 0) + (k & 3);
    const double2* Sp = reinterpret_cast<const double2*>(S) + cell0 + (size_t)m * cstride;
    double2 fn = Sp[0], fs = Sp[KG];
    { const double2 e = fn, o = fs; fn = cadd(e, o); fs = csub(e, o); }       // stored as (even, odd) sums
    if (comp == 1) { fn = make_double2(fn.y, -fn.x); fs = make_double2(fs.y, -fs.x); }
    double2 ph = make_double2(1.0, 0.0);
    if (shift) { ph = __ldg(tw2 + m % (2 * N)); ph.y = -ph.y; }
    const double w = (m == 0) ? 0.5 : 1.0;
    double2 dn = cmul(ph, fn), ds = cmul(ph, fs);
    dn.x *= w; dn.y *= w; ds.x *= w; ds.y *= w;
    const int b = m % N;
    const bool selfc = b == 0 || 2 * b == N;              // the bin is its own conjugate: both passes of the assembly hit it
    const int bb = 2 * b > N ? N - b : b;
    double2 yn, ys;
    if (selfc) { yn = make_double2(2.0 * dn.x, 0.0); ys = make_double2(2.0 * ds.x, 0.0); }
    else if (2 * b < N) { yn = dn; ys = ds; }
    else { yn = make_double2(dn.x, -dn.y); ys = make_double2(ds.x, -ds.y); }
    if (equator) ys = make_double2(0.0, 0.0);
    const double scale = 4.0 * 3.14159265358979323846 / (double)d.npix * (double)N;
    double2* Rp = reinterpret_cast<double2*>(R) + cell0;
    for (int pass = 0; pass < (selfc ? 1 : 2); ++pass) {
        double2 tn = yn, ts = ys;
        if (pass == 1) { tn.y = -tn.y; ts.y = -ts.y; }
        for (int mm = pass == 0 ? bb : N - bb; mm < mlim; mm += N) {
            double2 p2 = make_double2(scale, 0.0);
            if (shift) { p2 = __ldg(tw2 + mm % (2 * N)); p2.x *= scale; p2.y *= scale; }
            double2 se, so;
            if (equator) { se = cmul(p2, tn); so = make_double2(0.0, 0.0); }
            else { se = cmul(p2, cadd(tn, ts)); so = cmul(p2, csub(tn, ts)); }
            if (comp == 1) { se = make_double2(-se.y, se.x); so = make_double2(-so.y, so.x); }
            double2* c = Rp + (size_t)mm * cstride;
            c[0] = csub(c[0], se);
            c[KG] = csub(c[KG], so);
        }
    }
}

__global__ void __launch_bounds__(128) k_gs_update(DevicePlan d, const double* __restrict__ S, double* __restrict__ R, int m0, int kmaps, int p0)
{
    // one thread per (ring pair, map); the orders of one launch never share a bin
    gs_update_cell(d, S, R, p0 + blockIdx.y, blockIdx.z % d.ncomp, m0 + blockIdx.z / d.ncomp, blockIdx.x * blockDim.x + threadIdx.x, kmaps);
}

// The same correction for ALL orders of the ring pairs p >= pstar in one launch (hybrid sweep of Alg. 3): on a ring pair
// with mlim - 1 <= N / 2 no two orders share a bin, so the orders are independent there.  One thread per (order, map of
// the 4-map group): a warp walks 8 consecutive orders of one (ring pair, group), whose cells are consecutive 128-byte lines.
__global__ void __launch_bounds__(128) k_gs_update_free(DevicePlan d, const double* __restrict__ S, double* __restrict__ R, int pstar, int kmaps)
{
    const int p = pstar + blockIdx.y, comp = blockIdx.z % d.ncomp, kg = blockIdx.z / d.ncomp;
    const int m = blockIdx.x * 32 + (threadIdx.x >> 2), k = kg * KG + (threadIdx.x & 3);
    if (m > d.lmax) return;
    gs_update_cell(d, S, R, p, comp, m, k, kmaps);
}

// alm (rows from k0) += da (rows from 0) at the orders m >= m0: the m-major layout makes them the tail of every row
__global__ void __launch_bounds__(256) k_alm_add_from(double2* __restrict__ alm, const double2* __restrict__ da, long long nalm, long long off0,
                                                      int k0, int nrow_per_map)
{
    const long long row = blockIdx.y;                          // map * ncomp + comp, from the chunk start
    double2* a = alm + ((long long)k0 * nrow_per_map + row) * nalm;
    const double2* b = da + row * nalm;
    for (long long i = off0 + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nalm; i += (long long)gridDim.x * blockDim.x) {
        double2 v = a[i];
        const double2 w = b[i];
        v.x += w.x; v.y += w.y;
        a[i] = v;
    }
}

// sum of squares of the residual pixels from R by Parseval (the accumulation of k_ring_residual on its own):
// acc[k][comp] += (1/N) (sum over the orders m <= N/2, m < mlim of w |R_m|^2 / d sigma^2 + upow)
__global__ void __launch_bounds__(128) k_ring_power(DevicePlan d, const double* __restrict__ R, const double* __restrict__ upow,
                                                    double* __restrict__ acc_out, int kmaps)
{
    const int p = blockIdx.y, comp = blockIdx.z;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= kmaps) return;
    const RingPair& rp = d.rings[p];
    const int N = rp.n;
    const bool equator = rp.start_s < 0;
    const int mend = min(rp.mlim, N / 2 + 1);
    const size_t cstride = (size_t)d.ncomp * 2 * KG;
    const double2* Rp = reinterpret_cast<const double2*>(R) + f_cell(d, p, k >> 2, 0, comp, 0) + (k & 3);
    double ssq = 0.0;
    for (int m = 0; m < mend; ++m, Rp += cstride) {
        const double2 E = Rp[0], O = Rp[KG];
        const double w = (m == 0 || 2 * m == N) ? 1.0 : 2.0;
        const double q = equator ? (E.x * E.x + E.y * E.y) : 0.5 * (E.x * E.x + E.y * E.y + O.x * O.x + O.y * O.y);
        ssq = fma(w, q, ssq);
    }
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    const double tot = ssq / (dsig * dsig) + upow[((size_t)p * d.ncomp + comp) * d.kpad + k];
    if (tot != 0.0) atomicAdd(acc_out + (size_t)k * d.ncomp + comp, tot / (double)N);
}

// CTAs that share an SM with another one run RING_THREADS threads; a CTA that owns the SM runs twice as many
static int ring_threads(size_t smem) { return smem <= (size_t)113 * 1024 ? RING_THREADS : 2 * RING_THREADS; }

static cudaError_t ring_attr(sht_plan_s* pl)
{
    // the attribute belongs to the (function, device) pair: remembered per plan (a plan lives on one device)
    if (pl->ring_attr_set) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_ring_analysis, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_ring_synthesis, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
    if (e == cudaSuccess) pl->ring_attr_set = true;
    return e;
}

cudaError_t launch_ring_analysis(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st,
                                 double* upow)
{
    cudaError_t e = ring_attr(pl);
    if (e != cudaSuccess) return e;
    // the belt (two thirds of the pixels) and the cap rings on the chirp-z path go through the kernels of
    // sht_ring_pow2.cu, except when the uncovered power is wanted
    const bool fast = upow == nullptr && pl->fast_ring;
    if (fast && pl->belt_logn && (e = launch_ring_analysis_belt(pl, d, maps, F, k0, kmaps, st)) != cudaSuccess) return e;
    if (fast && (e = launch_ring_analysis_cz(pl, d, maps, F, k0, kmaps, st)) != cudaSuccess) return e;
    if (fast && (e = launch_ring_analysis_mr(pl, d, maps, F, k0, kmaps, st)) != cudaSuccess) return e;
    int* const* lists = fast ? pl->class_rings_nb : pl->class_rings;
    const int* count = fast ? pl->class_count_nb : pl->class_count;
    const int* ktmin = fast ? pl->class_ktmin_nb : pl->class_ktmin;
    // longest rings first: their CTAs are the slowest
    for (int c = RING_NCLASS - 1; c >= 0; --c) {
        if (count[c] == 0) continue;
        dim3 grid((kmaps + ktmin[c] - 1) / ktmin[c], count[c], d.ncomp);
        k_ring_analysis<<<grid, ring_threads(pl->class_smem[c]), pl->class_smem[c], st>>>(d, lists[c], maps, F, k0, kmaps, upow);
        pl->launches++;
    }
    return cudaGetLastError();
}

cudaError_t launch_ring_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps,
                                  const double* sub_from, int ksub0, cudaStream_t st)
{
    cudaError_t e = ring_attr(pl);
    if (e != cudaSuccess) return e;
    const bool fast = sub_from == nullptr && pl->fast_ring;
    if (fast && pl->belt_logn && (e = launch_ring_synthesis_belt(pl, d, F, maps, k0, kmaps, st)) != cudaSuccess) return e;
    if (fast && (e = launch_ring_synthesis_cz(pl, d, F, maps, k0, kmaps, st)) != cudaSuccess) return e;
    if (fast && (e = launch_ring_synthesis_mr(pl, d, F, maps, k0, kmaps, st)) != cudaSuccess) return e;
    int* const* lists = fast ? pl->class_rings_nb : pl->class_rings;
    const int* count = fast ? pl->class_count_nb : pl->class_count;
    const int* ktmin = fast ? pl->class_ktmin_nb : pl->class_ktmin;
    for (int c = RING_NCLASS - 1; c >= 0; --c) {
        if (count[c] == 0) continue;
        dim3 grid((kmaps + ktmin[c] - 1) / ktmin[c], count[c], d.ncomp);
        k_ring_synthesis<<<grid, ring_threads(pl->class_smem[c]), pl->class_smem[c], st>>>(d, lists[c], F, maps, k0, kmaps, sub_from, ksub0);
        pl->launches++;
    }
    return cudaGetLastError();
}

// residual of one Jacobi round in T_m-space: F (synthesised, north / south) <- Fmap - alias(F), folded; acc[k][comp] +=
// sum of squares of the residual pixels
cudaError_t launch_ring_residual(sht_plan_s* pl, const DevicePlan& d, double* F, const double* Fmap, const double* upow, double* acc,
                                 int kmaps, cudaStream_t st)
{
    cudaError_t e = ring_attr(pl);
    if (e == cudaSuccess && !pl->resid_attr_set) {
        e = cudaFuncSetAttribute(k_ring_residual, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
        pl->resid_attr_set = e == cudaSuccess;
    }
    if (e != cudaSuccess) return e;
    for (int c = RING_NCLASS - 1; c >= 0; --c) {
        if (pl->class_count[c] == 0) continue;
        dim3 grid((kmaps + pl->class_ktmin[c] - 1) / pl->class_ktmin[c], pl->class_count[c], d.ncomp);
        k_ring_residual<<<grid, ring_threads(pl->class_smem[c]), pl->class_smem[c] + 512, st>>>(d, pl->class_rings[c], F, Fmap, upow, acc, kmaps);
        pl->launches++;
    }
    return cudaGetLastError();
}

cudaError_t launch_gs_update(sht_plan_s* pl, const DevicePlan& d, const double* S, double* R, int m, int nm, int kmaps, cudaStream_t st, int np,
                             int p0)
{
    const int pend = np > 0 && np < d.nh ? np : d.nh;
    if (pend <= p0 || nm <= 0) return cudaSuccess;
    k_gs_update<<<dim3((unsigned)((kmaps + 127) / 128), (unsigned)(pend - p0), (unsigned)(nm * d.ncomp)), 128, 0, st>>>(d, S, R, m, kmaps, p0);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_gs_update_free(sht_plan_s* pl, const DevicePlan& d, const double* S, double* R, int pstar, int kmaps, cudaStream_t st)
{
    if (pstar >= d.nh) return cudaSuccess;
    const int nkg = (kmaps + KG - 1) / KG;
    k_gs_update_free<<<dim3((unsigned)((d.lmax + 32) / 32), (unsigned)(d.nh - pstar), (unsigned)(nkg * d.ncomp)), 128, 0, st>>>(d, S, R, pstar, kmaps);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_alm_add_from(sht_plan_s* pl, const DevicePlan& d, double* alm, const double* da, int k0, int kmaps, int m0, cudaStream_t st)
{
    if (m0 > d.lmax) return cudaSuccess;
    const long long off0 = (long long)m0 * (2 * d.lmax + 1 - m0) / 2 + m0;      // idx(l = m0, m0): first entry of order m0
    const long long n = d.nalm - off0;
    const unsigned gx = (unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024);
    k_alm_add_from<<<dim3(gx, (unsigned)(kmaps * d.ncomp)), 256, 0, st>>>(reinterpret_cast<double2*>(alm), reinterpret_cast<const double2*>(da),
                                                                        d.nalm, off0, k0, d.ncomp);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_ring_power(sht_plan_s* pl, const DevicePlan& d, const double* R, const double* upow, double* acc, int kmaps, cudaStream_t st)
{
    k_ring_power<<<dim3((unsigned)((kmaps + 127) / 128), (unsigned)d.nh, (unsigned)d.ncomp), 128, 0, st>>>(d, R, upow, acc, kmaps);
    pl->launches++;
    return cudaGetLastError();
}

}  // namespace sht
