// sht_ring_pow2.cu -- subsystem (1), fast path for the equatorial belt: the 2 nside + 1 rings of 4 nside pixels hold two
// thirds of all pixels, and for nside a power of two their length N = 4 nside is a power of two.
//
// Same mathematics as sht_ring_fft.cu (eq. 2 row 3 and App. A.1 :412-416 for the analysis side,
// :66-70 eq. 4 and :78 for the synthesis side); what differs is how the bytes move and how the transform is laid out:
//   * persistent CTAs (one per SM) loop over work items (ring pair, component, KT maps);
//   * analysis input: the map rows of the next items are fetched by 1-D bulk copies (cp.async.bulk, mbarrier
//     complete_tx) into a double-buffered staging area while the current item is transformed; analysis output: the
//     folded T_m lines are staged in shared memory and written by tiled TMA stores (cp.async.bulk.tensor) -- no thread
//     ever waits on a global load or issues a global store;
//   * synthesis input: the T_m lines arrive by tiled TMA loads through a ring of shared-memory slots;
//   * the length-N transform is compiled for its length (N = R1 R2 R3, radices 16 / 8, three passes in registers, no
//     divisions, no runtime radix list) as decimation in time on the analysis side -- first pass straight from the
//     staged rows, bins come out in NATURAL order, so the FFT mapping reads shared memory contiguously -- and as the
//     exact adjoint network (decimation in frequency) on the synthesis side: bins go in in natural order, the last pass
//     writes the pixels of the two rings coalesced.
// The north and the south ring of a pair are the real and the imaginary part of one complex sequence, as in the
// general kernels.  Twiddles: one table value per butterfly, the other powers by multiplication.
#include "sht_ring_common.cuh"

namespace sht {

namespace p2 {


// multiply by exp(-+ 2 pi i k / 16), k compile-time (- forward, + if INV)
template <int K, bool INV>
__device__ __forceinline__ double2 mul_w16(double2 a)
{
    constexpr int k = K & 15;
    constexpr double C1 = 0.92387953251128675613, S1 = 0.38268343236508977173, H = 0.70710678118654752440;
    if constexpr (k == 0) return a;
    else if constexpr (k == 4) return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    else if constexpr (k == 8) return make_double2(-a.x, -a.y);
    else if constexpr (k == 12) return INV ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
    else {
        // w = c - i s (forward), c + i s (inverse), angle 2 pi k / 16
        constexpr double c = (k == 1 || k == 15) ? C1 : (k == 2 || k == 14) ? H : (k == 3 || k == 13) ? S1
                           : (k == 5 || k == 11) ? -S1 : (k == 6 || k == 10) ? -H : -C1;
        constexpr double s0 = (k == 1 || k == 7) ? S1 : (k == 2 || k == 6) ? H : (k == 3 || k == 5) ? C1
                            : (k == 9 || k == 15) ? -S1 : (k == 10 || k == 14) ? -H : -C1;       // sin(2 pi k / 16)
        constexpr double sn = INV ? s0 : -s0;                                                 // imaginary part of w
        return make_double2(fma(a.x, c, -(a.y * sn)), fma(a.x, sn, a.y * c));
    }
}

// multiply by exp(-+ 2 pi i k / 12), k in {1, 2, 3, 4, 6}
template <int K, bool INV>
__device__ __forceinline__ double2 mul_w12(double2 a)
{
    constexpr double C30 = 0.86602540378443864676;       // cos(pi / 6)
    if constexpr (K == 3) return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
    else if constexpr (K == 6) return make_double2(-a.x, -a.y);
    else {
        constexpr double c = K == 1 ? C30 : K == 2 ? 0.5 : -0.5;                  // cos(2 pi K / 12)
        constexpr double s0 = K == 1 ? 0.5 : C30;                                // sin(2 pi K / 12), K = 1, 2, 4
        constexpr double sn = INV ? s0 : -s0;
        return make_double2(fma(a.x, c, -(a.y * sn)), fma(a.x, sn, a.y * c));
    }
}

template <bool INV>
__device__ __forceinline__ void bfly4(double2& x0, double2& x1, double2& x2, double2& x3)
{
    const double2 v0 = cadd(x0, x2), v1 = csub(x0, x2), v2 = cadd(x1, x3), dd = csub(x1, x3);
    const double2 v3 = INV ? make_double2(-dd.y, dd.x) : make_double2(dd.y, -dd.x);      // (-+ i)(x1 - x3)
    x0 = cadd(v0, v2); x1 = cadd(v1, v3); x2 = csub(v0, v2); x3 = csub(v1, v3);
}

// R-point DFT in registers, natural order in and out: u[k] <- sum_n u[n] exp(-+ 2 pi i n k / R)
template <int R, bool INV>
__device__ __forceinline__ void dft(double2 (&u)[R])
{
    static_assert(R == 8 || R == 12 || R == 16, "radix");
    if constexpr (R == 12) {
        // n = 4 n1 + n2, k = k1 + 3 k2:  X[k1 + 3 k2] = sum_n2 w4^{n2 k2} { w12^{n2 k1} sum_n1 x[4 n1 + n2] w3^{n1 k1} }
        constexpr double S3 = 0.86602540378443864676;    // sin(2 pi / 6)
        double2 t[4][3];
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) {
            const double2 x0 = u[n2], x1 = u[n2 + 4], x2 = u[n2 + 8];
            const double2 sm = cadd(x1, x2), df = csub(x1, x2);
            const double2 re = make_double2(fma(-0.5, sm.x, x0.x), fma(-0.5, sm.y, x0.y));
            // forward: X1 = re - i S3 df, X2 = re + i S3 df; inverse: the other way round
            const double2 im = make_double2(S3 * df.y, -S3 * df.x);              // -i S3 df
            double2 y1 = INV ? csub(re, im) : cadd(re, im), y2 = INV ? cadd(re, im) : csub(re, im);
            // twiddle w12^{n2 k1}: exponents n2 (k1 = 1), 2 n2 (k1 = 2)
            if (n2 == 1) { y1 = mul_w12<1, INV>(y1); y2 = mul_w12<2, INV>(y2); }
            if (n2 == 2) { y1 = mul_w12<2, INV>(y1); y2 = mul_w12<4, INV>(y2); }
            if (n2 == 3) { y1 = mul_w12<3, INV>(y1); y2 = mul_w12<6, INV>(y2); }
            t[n2][0] = cadd(x0, sm); t[n2][1] = y1; t[n2][2] = y2;
        }
#pragma unroll
        for (int k1 = 0; k1 < 3; ++k1) {
            double2 w0 = t[0][k1], w1 = t[1][k1], w2 = t[2][k1], w3 = t[3][k1];
            bfly4<INV>(w0, w1, w2, w3);
            u[k1] = w0; u[k1 + 3] = w1; u[k1 + 6] = w2; u[k1 + 9] = w3;
        }
    } else if constexpr (R == 16) {
        // n = a + 4 r, k = s + 4 q:  X[s + 4 q] = sum_a w4^{a q} { w16^{a s} sum_r x[a + 4 r] w4^{r s} }
        double2 t[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            double2 v0 = u[a], v1 = u[a + 4], v2 = u[a + 8], v3 = u[a + 12];
            bfly4<INV>(v0, v1, v2, v3);
            t[a][0] = v0;
            t[a][1] = a == 0 ? v1 : a == 1 ? mul_w16<1, INV>(v1) : a == 2 ? mul_w16<2, INV>(v1) : mul_w16<3, INV>(v1);
            t[a][2] = a == 0 ? v2 : a == 1 ? mul_w16<2, INV>(v2) : a == 2 ? mul_w16<4, INV>(v2) : mul_w16<6, INV>(v2);
            t[a][3] = a == 0 ? v3 : a == 1 ? mul_w16<3, INV>(v3) : a == 2 ? mul_w16<6, INV>(v3) : mul_w16<9, INV>(v3);
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            double2 w0 = t[0][s], w1 = t[1][s], w2 = t[2][s], w3 = t[3][s];
            bfly4<INV>(w0, w1, w2, w3);
            u[s] = w0; u[s + 4] = w1; u[s + 8] = w2; u[s + 12] = w3;
        }
    } else {
        // n = a + 2 r, k = s + 4 q:  X[s + 4 q] = sum_a (-1)^{a q} { w8^{a s} sum_r x[a + 2 r] w4^{r s} }
        double2 e0 = u[0], e1 = u[2], e2 = u[4], e3 = u[6];
        double2 o0 = u[1], o1 = u[3], o2 = u[5], o3 = u[7];
        bfly4<INV>(e0, e1, e2, e3);
        bfly4<INV>(o0, o1, o2, o3);
        o1 = mul_w16<2, INV>(o1); o2 = mul_w16<4, INV>(o2); o3 = mul_w16<6, INV>(o3);
        u[0] = cadd(e0, o0); u[4] = csub(e0, o0);
        u[1] = cadd(e1, o1); u[5] = csub(e1, o1);
        u[2] = cadd(e2, o2); u[6] = csub(e2, o2);
        u[3] = cadd(e3, o3); u[7] = csub(e3, o3);
    }
}

// u[k] *= w^k, k = 1 .. R-1: the powers by multiplication, w^{4 i + r} = (w^4)^i w^r with w, w^2, w^3 and the running
// (w^4)^i kept (few live registers; dependency depth <= 5 complex products)
template <int R>
__device__ __forceinline__ void mul_powers(double2 (&u)[R], double2 w)
{
    static_assert(R % 4 == 0, "radix");
    const double2 w2 = cmul(w, w), w3 = cmul(w2, w);
    u[1] = cmul(u[1], w); u[2] = cmul(u[2], w2); u[3] = cmul(u[3], w3);
    double2 b = cmul(w2, w2);                             // w^4
#pragma unroll
    for (int i = 1; i < R / 4; ++i) {
        u[4 * i] = cmul(u[4 * i], b);
        u[4 * i + 1] = cmul(u[4 * i + 1], cmul(b, w));
        u[4 * i + 2] = cmul(u[4 * i + 2], cmul(b, w2));
        u[4 * i + 3] = cmul(u[4 * i + 3], cmul(b, w3));
        if (i + 1 < R / 4) b = (i == 1) ? cmul(b, b) : cmul(b, cmul(w2, w2));     // w^8 = (w^4)^2, w^12 = w^8 w^4
    }
}

// transform geometry of a ring length N = 2^LOGN = R1 R2 R3
template <int LOGN>
struct Geo {
    static constexpr int N = 1 << LOGN;
    static constexpr int R1 = LOGN >= 10 ? 16 : 8;       // 512 = 8.8.8, 1024 = 16.8.8, 2048 = 16.16.8, 4096 = 16.16.16
    static constexpr int R2 = LOGN >= 11 ? 16 : 8;
    static constexpr int R3 = LOGN >= 12 ? 16 : 8;
    static constexpr int LR1 = R1 == 16 ? 4 : 3, LR2 = R2 == 16 ? 4 : 3, LR3 = R3 == 16 ? 4 : 3;
    static_assert(R1 * R2 * R3 == N, "radix split");
    // shared-memory position of element p: one element of padding per R1 and one more per R1 R2 elements makes all
    // three passes free of bank conflicts (16-byte elements, quarter-warp phases)
    static constexpr int NPAD = N + N / R1 + N / (R1 * R2);
    __device__ static __forceinline__ int phys(int p) { return p + (p >> LR1) + (p >> (LR1 + LR2)); }
};

// per-map buffer stride (elements): = 8 / KT mod 8, so that the KT maps a quarter-warp touches in the FFT mapping fall
// into different bank groups
template <int LOGN, int KT>
__host__ __device__ constexpr int buf_stride()
{
    constexpr int np = Geo<LOGN>::NPAD, want = (8 / KT) & 7;
    return np + ((want - (np & 7)) & 7);
}

constexpr int NT = 256;                                  // threads per CTA (one CTA per SM)

// work item -> (ring pair, component, first map of the KT maps)
struct Item {
    int p, comp, kfirst;
};
__device__ __forceinline__ Item decode_item(long long it, int nkp, int ncomp, int p_first, int kt)
{
    const int kp = (int)(it % nkp);
    const long long r = it / nkp;
    Item o;
    o.comp = (int)(r % ncomp);
    o.p = p_first + (int)(r / ncomp);
    o.kfirst = kp * kt;
    return o;
}

}  // namespace p2

// ------------------------------------------------------------------------------------------------
// analysis: maps -> F for the belt ring pairs p_first .. p_first + npairs - 1 (all of length N = 2^LOGN), two CTAs per
// SM.  The rows of an item are bulk-copied straight into the transform buffers; every thread owns exactly one pass-A
// butterfly, reads its inputs into registers, and the pass writes the buffers in place after a barrier.  There is no
// prefetch inside a CTA: the copy of the next item is in flight while the OTHER CTA of the SM computes (a variant with
// a double-buffered input staging area and one CTA per SM had half the warps and was 15 % slower).
// shared memory: [KT transform buffers][4 output slots][mbarrier]
// ------------------------------------------------------------------------------------------------
template <int LOGN, int KT>
__global__ void __launch_bounds__(p2::NT, 2)
k_ring_analysis_p2i(const __grid_constant__ CUtensorMap tmF, DevicePlan d, const double* __restrict__ maps, int k0, int kmaps,
                    int p_first, int npairs, int planes)
{
    using namespace p2;
    using G = Geo<LOGN>;
    constexpr int N = G::N, R1 = G::R1, R2 = G::R2, R3 = G::R3;
    constexpr int TPM = NT / KT, MB = NT / KT;
    constexpr int BS = buf_stride<LOGN, KT>();
    constexpr int SLOT = MB * 2 * KT, NSLOTS = 4, U = 2;
    static_assert(N / R1 <= TPM, "one pass-A butterfly per thread");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* tr = reinterpret_cast<double2*>(smem_raw);
    double2* ostage = tr + KT * BS;
    uint64_t* full = reinterpret_cast<uint64_t*>(ostage + NSLOTS * SLOT);

    const int tid = threadIdx.x;
    const int nkp = (kmaps + KT - 1) / KT;
    const long long nitems = (long long)npairs * d.ncomp * nkp;
    const int out_hs = planes ? MB : 1, out_ms = planes ? 1 : 2;
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    if (tid == 0) {
        mbar_init(full, 1);
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();
    auto issue_loads = [&](long long it) {
        const Item w = decode_item(it, nkp, d.ncomp, p_first, KT);
        const RingPair& rp = d.rings[w.p];
        const bool eq = rp.start_s < 0;
        mbar_arrive_expect_tx(full, (uint32_t)(KT * (eq ? 1 : 2) * N * 8));
#pragma unroll
        for (int kk = 0; kk < KT; ++kk) {
            const int k = min(w.kfirst + kk, kmaps - 1);
            const double* mp = maps + ((size_t)(k0 + k) * d.ncomp + w.comp) * d.npix;
            double* dst = reinterpret_cast<double*>(tr + kk * BS);
            bulk_load(dst, mp + rp.start_n, N * 8, full);
            if (!eq) bulk_load(dst + N, mp + rp.start_s, N * 8, full);
        }
    };
    if (tid == 0 && (long long)blockIdx.x < nitems) issue_loads(blockIdx.x);

    const int kkp = tid / TPM, tm = tid - kkp * TPM;
    const int kkm = tid & (KT - 1), mi = tid / KT;
    // per-thread constants of the whole launch (every belt ring has the same length): pass twiddles W_N^j, W_N^{R1 n2'},
    // and the phase recurrence of the FFT mapping, W_{2N}^{mi} d sigma and W_{2N}^{MB}
    constexpr int NIA = (N / R1 + TPM - 1) / TPM, NIB = (N / R2 + TPM - 1) / TPM;
    const double2* __restrict__ twc = d.tw + d.rings[p_first].tw_off;
    double2 twA[NIA], twB[NIB];
#pragma unroll
    for (int i = 0; i < NIA; ++i) twA[i] = __ldg(twc + 2 * ((tm + i * TPM) & (N / R1 - 1)));
#pragma unroll
    for (int i = 0; i < NIB; ++i) twB[i] = __ldg(twc + 2 * R1 * (((tm + i * TPM) & (N / R2 - 1)) >> G::LR1));
    double2 ph0 = __ldg(twc + (mi & (2 * N - 1)));
    ph0.x *= dsig; ph0.y *= dsig;
    const double2 phs = __ldg(twc + (MB & (2 * N - 1)));
    int li = 0, nstore = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x, ++li) {
        const Item w = decode_item(it, nkp, d.ncomp, p_first, KT);
        const RingPair rp = d.rings[w.p];
        const bool equator = rp.start_s < 0;
        mbar_wait(full, li & 1);
        double2* trk = tr + kkp * BS;
        // ---- pass A in place: inputs to registers, barrier, transform, write
        {
            const int j = tm;
            const bool act = j < N / R1;
            double2 u[R1];
            if (act) {
                const double* rows = reinterpret_cast<const double*>(trk);
#pragma unroll
                for (int r = 0; r < R1; ++r) {
                    u[r].x = rows[j + r * (N / R1)];
                    u[r].y = equator ? 0.0 : rows[N + j + r * (N / R1)];
                }
            }
            __syncthreads();
            if (act) {
                dft<R1, false>(u);
                mul_powers<R1>(u, twA[0]);
                const int B = (j >> G::LR3) + R2 * (j & (R3 - 1));
                double2* dst = trk + R1 * B + B + (j & (R3 - 1));
#pragma unroll
                for (int k = 0; k < R1; ++k) dst[k] = u[k];
            }
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < NIB; ++i) {
            const int wq = tm + i * TPM;
            if (wq >= N / R2) break;
            const int k1 = wq & (R1 - 1), n2p = wq >> G::LR1;
            double2* base = trk + k1 + (R1 * R2 + R2 + 1) * n2p;
            double2 u[R2];
#pragma unroll
            for (int t = 0; t < R2; ++t) u[t] = base[(R1 + 1) * t];
            dft<R2, false>(u);
            mul_powers<R2>(u, twB[i]);
#pragma unroll
            for (int t = 0; t < R2; ++t) base[(R1 + 1) * t] = u[t];
        }
        __syncthreads();
        for (int wq = tm; wq < N / R3; wq += TPM) {
            const int k1 = wq & (R1 - 1), k1p = wq >> G::LR1;
            double2* base = trk + k1 + (R1 + 1) * k1p;
            double2 u[R3];
#pragma unroll
            for (int t = 0; t < R3; ++t) u[t] = base[(R1 * R2 + R2 + 1) * t];
            dft<R3, false>(u);
#pragma unroll
            for (int t = 0; t < R3; ++t) base[(R1 * R2 + R2 + 1) * t] = u[t];
        }
        __syncthreads();
        // ---- FFT mapping, U boxes per round through a ring of NSLOTS output slots
        const int mlim = rp.mlim;
        const double2* trm = tr + kkm * BS;
        const int kg = w.kfirst / KG, csel = (w.kfirst % KG) / KT;
        double2 phc = rp.shift ? ph0 : make_double2(dsig, 0.0);
        const double2 pstep = rp.shift ? phs : make_double2(1.0, 0.0);
        for (int m0 = 0; m0 < mlim; m0 += U * MB) {
#pragma unroll
            for (int q = 0; q < U; ++q) {
                const int m = m0 + q * MB + mi;
                const int b = m & (N - 1), bc = (N - b) & (N - 1);
                const double2 A = trm[G::phys(b)], Bv = trm[G::phys(bc)];
                const double2 gn = make_double2(0.5 * (A.x + Bv.x), 0.5 * (A.y - Bv.y));
                const double2 gs = make_double2(0.5 * (A.y + Bv.y), -0.5 * (A.x - Bv.x));
                const double2 ph = phc;                   // d sigma e^{-i m phi0}, phi0 = pi / N on the shifted rings
                phc = cmul(phc, pstep);
                double2 E, O;
                if (equator) { E = cmul(ph, gn); O = make_double2(0.0, 0.0); }
                else { E = cmul(ph, cadd(gn, gs)); O = cmul(ph, csub(gn, gs)); }
                if (w.comp == 1) { E = make_double2(-E.y, E.x); O = make_double2(-O.y, O.x); }
                double2* slot = ostage + ((nstore + q) % NSLOTS) * SLOT;
                slot[(mi * out_ms) * KT + kkm] = E;
                slot[(out_hs + mi * out_ms) * KT + kkm] = O;
            }
            fence_async_smem();
            if (tid == 0) bulk_wait_read<0>();
            __syncthreads();
            if (tid == 0) {
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    const int mq = m0 + q * MB;
                    if (mq >= mlim) break;
                    const double2* slot = ostage + ((nstore + q) % NSLOTS) * SLOT;
                    if (planes) tma_store_5d(&tmF, slot, 0, mq, 2 * w.comp, csel, w.p * d.nkg + kg);
                    else tma_store_5d(&tmF, slot, 0, csel, 2 * w.comp, mq, w.p * d.nkg + kg);
                }
                bulk_commit();
            }
            nstore += U;
        }
        // every thread has passed the last round's barrier, i.e. finished reading the transform buffers
        if (tid == 0 && it + gridDim.x < nitems) issue_loads(it + gridDim.x);
    }
    if (tid == 0) bulk_wait<0>();
}

// ------------------------------------------------------------------------------------------------
// synthesis: F (even / odd sums of the Legendre synthesis) -> maps for the belt ring pairs.
// shared memory: [KT transform buffers][NSL input slots of MB orders][mbarriers]
// The ring spectrum of the packed sequence z = north + i south is accumulated cell by cell: order m adds
// (w_m / 2)(d_n + i d_s) to bin m mod N and (w_m / 2)(conj d_n + i conj d_s) to bin -m mod N, d = e^{+i m phi0} T_m
// (eq. 4; at the self-conjugate bins 0 and N/2 the two add up to the real parts, reading G8).
// ------------------------------------------------------------------------------------------------
template <int LOGN, int KT, int NSL>
__global__ void __launch_bounds__(p2::NT, 2)
k_ring_synthesis_p2(const __grid_constant__ CUtensorMap tmF, DevicePlan d, double* __restrict__ maps, int k0, int kmaps,
                    int p_first, int npairs, int planes)
{
    using namespace p2;
    using G = Geo<LOGN>;
    constexpr int N = G::N, R1 = G::R1, R2 = G::R2, R3 = G::R3;
    constexpr int TPM = NT / KT, MB = NT / KT;
    constexpr int BS = buf_stride<LOGN, KT>();
    constexpr int SLOT = MB * 2 * KT;                     // double2 per input slot
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* in_slots = reinterpret_cast<double2*>(smem_raw);
    double2* tr = in_slots + NSL * SLOT;
    uint64_t* full = reinterpret_cast<uint64_t*>(tr + KT * BS);

    const int tid = threadIdx.x;
    const int nkp = (kmaps + KT - 1) / KT;
    const long long nitems = (long long)npairs * d.ncomp * nkp;
    const int in_hs = planes ? MB : 1, in_ms = planes ? 1 : 2;
    if (tid == 0) {
        for (int s = 0; s < NSL; ++s) mbar_init(full + s, 1);
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();

    // producer state (thread 0): the flattened sequence of (item, chunk) this CTA consumes, NSL chunks ahead
    long long pit = blockIdx.x;
    int pm0 = 0, pmlim = 0, pslot = 0;
    Item pw{0, 0, 0};
    auto producer_begin_item = [&]() {
        if (pit < nitems) { pw = decode_item(pit, nkp, d.ncomp, p_first, KT); pmlim = d.rings[pw.p].mlim; pm0 = 0; }
    };
    auto produce_one = [&]() {                            // issue the next chunk if there is one
        if (pit >= nitems) return;
        mbar_arrive_expect_tx(full + pslot, SLOT * 16);
        const int kg = pw.kfirst / KG, csel = (pw.kfirst % KG) / KT;
        if (planes) tma_load_5d(in_slots + pslot * SLOT, &tmF, full + pslot, 0, pm0, 2 * pw.comp, csel, pw.p * d.nkg + kg);
        else tma_load_5d(in_slots + pslot * SLOT, &tmF, full + pslot, 0, csel, 2 * pw.comp, pm0, pw.p * d.nkg + kg);
        pslot = pslot + 1 == NSL ? 0 : pslot + 1;
        pm0 += MB;
        if (pm0 >= pmlim) { pit += gridDim.x; producer_begin_item(); }
    };
    if (tid == 0) {
        producer_begin_item();
        for (int s = 0; s < NSL; ++s) produce_one();
    }

    const int kkp = tid / TPM, tm = tid - kkp * TPM;
    const int kkm = tid & (KT - 1), mi = tid / KT;
    // per-thread constants of the whole launch: conjugate pass twiddles, and the phase recurrence of the inverse mapping
    constexpr int NIA = (N / R1 + TPM - 1) / TPM, NIC = (N / R3 + TPM - 1) / TPM;
    const double2* __restrict__ twc = d.tw + d.rings[p_first].tw_off;
    double2 twA[NIA], twC[NIC];
#pragma unroll
    for (int i = 0; i < NIA; ++i) { twA[i] = __ldg(twc + 2 * ((tm + i * TPM) & (N / R1 - 1))); twA[i].y = -twA[i].y; }
#pragma unroll
    for (int i = 0; i < NIC; ++i) { twC[i] = __ldg(twc + 2 * R1 * (((tm + i * TPM) & (N / R3 - 1)) >> G::LR1)); twC[i].y = -twC[i].y; }
    double2 ph0 = __ldg(twc + (mi & (2 * N - 1)));       // e^{+i mi phi0}
    ph0.y = -ph0.y;
    double2 phs = __ldg(twc + (MB & (2 * N - 1)));
    phs.y = -phs.y;
    int cslot = 0; uint32_t cphase = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x) {
        const Item w = decode_item(it, nkp, d.ncomp, p_first, KT);
        const RingPair rp = d.rings[w.p];
        const bool equator = rp.start_s < 0;
        for (int i = tid; i < KT * BS; i += NT) tr[i] = make_double2(0.0, 0.0);
        __syncthreads();
        // ---- inverse FFT mapping: accumulate the ring spectrum
        const int mlim = rp.mlim;
        double2* trm = tr + kkm * BS;
        double2 phc = rp.shift ? ph0 : make_double2(1.0, 0.0);
        const double2 pstep = rp.shift ? phs : make_double2(1.0, 0.0);
        for (int m0 = 0; m0 < mlim; m0 += MB) {
            mbar_wait(full + cslot, cphase);
            const double2* slot = in_slots + cslot * SLOT;
            const int m = m0 + mi;
            const bool live = m < mlim;
            double2 zd = make_double2(0.0, 0.0), zc = zd;
            if (live) {
                const double2 e = slot[(mi * in_ms) * KT + kkm], o = slot[(in_hs + mi * in_ms) * KT + kkm];
                double2 fn = cadd(e, o), fs = csub(e, o);                        // stored as (even, odd) sums
                if (w.comp == 1) { fn = make_double2(fn.y, -fn.x); fs = make_double2(fs.y, -fs.x); }   // U = -i (iU)
                if (equator) fs = make_double2(0.0, 0.0);
                double2 ph = phc;
                const double wgt = (m == 0) ? 0.5 : 1.0;
                ph.x *= wgt; ph.y *= wgt;
                const double2 dn = cmul(ph, fn), ds = cmul(ph, fs);
                zd = make_double2(dn.x - ds.y, dn.y + ds.x);                     // d_n + i d_s
                zc = make_double2(dn.x + ds.y, ds.x - dn.y);                     // conj d_n + i conj d_s
            }
            phc = cmul(phc, pstep);
            const int b1 = m & (N - 1), b2 = (N - b1) & (N - 1);
            // two orders of one chunk meet in a bin only if m + m' = 0 mod N for some pair of the chunk
            const bool clash = ((2 * m0 + N - 1) / N) * N <= 2 * m0 + 2 * MB - 2;
            if (live) { double2* c1 = trm + G::phys(b1); *c1 = cadd(*c1, zd); }
            if (clash) __syncthreads();
            if (live) { double2* c2 = trm + G::phys(b2); *c2 = cadd(*c2, zc); }
            __syncthreads();                              // slot consumed (and bins of this chunk settled)
            if (tid == 0) produce_one();
            if (++cslot == NSL) { cslot = 0; cphase ^= 1; }
        }
        double2* trk = tr + kkp * BS;
        // ---- pass C^-1: inverse R3-point transforms over k2', then the conjugate twiddle W_{R2 R3}^{-n2' k1'}
#pragma unroll
        for (int i = 0; i < NIC; ++i) {
            const int wq = tm + i * TPM;
            if (wq >= N / R3) break;
            const int k1 = wq & (R1 - 1), k1p = wq >> G::LR1;
            double2* base = trk + k1 + (R1 + 1) * k1p;
            double2 u[R3];
#pragma unroll
            for (int t = 0; t < R3; ++t) u[t] = base[(R1 * R2 + R2 + 1) * t];
            dft<R3, true>(u);
            mul_powers<R3>(u, twC[i]);                    // conj W_N^{R1 k1'}: (W^{k1'})^{n2'}, n2' = t
#pragma unroll
            for (int t = 0; t < R3; ++t) base[(R1 * R2 + R2 + 1) * t] = u[t];
        }
        __syncthreads();
        // ---- pass B^-1: inverse R2-point transforms over k1' at positions k1 + R1 t + R1 R2 n2'
        for (int wq = tm; wq < N / R2; wq += TPM) {
            const int k1 = wq & (R1 - 1), n2p = wq >> G::LR1;
            double2* base = trk + k1 + (R1 * R2 + R2 + 1) * n2p;
            double2 u[R2];
#pragma unroll
            for (int t = 0; t < R2; ++t) u[t] = base[(R1 + 1) * t];
            dft<R2, true>(u);
#pragma unroll
            for (int t = 0; t < R2; ++t) base[(R1 + 1) * t] = u[t];
        }
        __syncthreads();
        // ---- pass A^-1: conjugate twiddle W_N^{-n2 k1}, inverse R1-point transforms over k1 -> pixels n1 N / R1 + n2
        const int k = w.kfirst + kkp;
        double* mp = maps + ((size_t)(k0 + (k < kmaps ? k : 0)) * d.ncomp + w.comp) * d.npix;
#pragma unroll
        for (int i = 0; i < NIA; ++i) {
            const int j = tm + i * TPM;
            if (j >= N / R1) break;
            const int B = (j >> G::LR3) + R2 * (j & (R3 - 1));
            const double2* src = trk + R1 * B + B + (j & (R3 - 1));
            double2 u[R1];
#pragma unroll
            for (int q = 0; q < R1; ++q) u[q] = src[q];
            mul_powers<R1>(u, twA[i]);
            dft<R1, true>(u);
            if (k < kmaps) {
#pragma unroll
                for (int r = 0; r < R1; ++r) {
                    mp[rp.start_n + j + r * (N / R1)] = u[r].x;
                    if (!equator) mp[rp.start_s + j + r * (N / R1)] = u[r].y;
                }
            }
        }
        __syncthreads();                                  // the transform buffers are rewritten by the next item
    }
}

// ================================================================================================
// Cap rings (length N = 4 i, any i) by the chirp-z transform (Bluestein) on top of the compiled transforms:
//   X_b = c_b sum_n (x_n c_n) h_{b-n},   c_j = exp(-i pi j^2 / N),  h = conj c,
// a circular convolution of a compiled length L >= 2 N - 1 (L = 2^a or 3 2^a): forward transform (decimation in time,
// natural-order spectrum), product with the plan's filter spectrum FFT_L(h) / L, inverse transform (the adjoint
// network), chirp.  The last forward pass, the filter product and the first inverse pass work on the same elements
// and are one pass in registers.  Data movement as for the belt: bulk copies in, TMA stores out, persistent CTAs.
// Per ring pair the plan holds [filter spectrum, natural order: L][chirp c_j: N] (cz table).
// ================================================================================================
namespace p2 {

template <int R1_, int R2_, int R3_>
struct GeoT {
    static constexpr int R1 = R1_, R2 = R2_, R3 = R3_, L = R1_ * R2_ * R3_;
    static constexpr int LR1 = R1 == 16 ? 4 : 3, LR2 = R2 == 16 ? 4 : 3;
    static_assert((R1 == 8 || R1 == 16) && (R2 == 8 || R2 == 16), "the first two radices are powers of two");
    static constexpr int S2 = R1 + 1, S3 = R1 * R2 + R2 + 1;          // physical strides of the second / third digit
    static constexpr int LPAD = L + L / R1 + L / (R1 * R2);
    __device__ static __forceinline__ int phys(int p) { return p + (p >> LR1) + (p >> (LR1 + LR2)); }
};

// forward passes B and the fused [C, filter, C^-1] pass, inverse pass B^-1 of one map's buffer; `tm`, `TPM`: thread
// inside the map / threads per map; twL[e] = W_L^e; hf: filter spectrum in natural order (CONJ: conjugated)
// per-thread twiddles of a chirp-z launch (the convolution length is the same for every ring of the launch):
// W_L^j of the butterflies the thread owns in pass A / A^-1, W_L^{R1 n2'} (pass B) and W_L^{R1 k1'} (fused pass)
template <class G, int TPM>
struct CzTw {
    static constexpr int NIA = (G::L / G::R1 + TPM - 1) / TPM, NIB = (G::L / G::R2 + TPM - 1) / TPM,
                         NIC = (G::L / G::R3 + TPM - 1) / TPM;
    double2 a[NIA], b[NIB], c[NIC];
    __device__ __forceinline__ void load(const double2* __restrict__ twL, int tm)
    {
#pragma unroll
        for (int i = 0; i < NIA; ++i) { const int j = tm + i * TPM; a[i] = __ldg(twL + (j < G::L / G::R1 ? j : 0)); }
#pragma unroll
        for (int i = 0; i < NIB; ++i) { const int w = tm + i * TPM; b[i] = __ldg(twL + (w < G::L / G::R2 ? G::R1 * (w >> G::LR1) : 0)); }
#pragma unroll
        for (int i = 0; i < NIC; ++i) { const int w = tm + i * TPM; c[i] = __ldg(twL + (w < G::L / G::R3 ? G::R1 * (w >> G::LR1) : 0)); }
    }
};

// forward pass B, the fused [C, filter, C^-1] pass and the inverse pass B^-1 on one map's buffer; `tm`: thread inside
// the map; hf: filter spectrum in natural order (CONJ: conjugated)
template <class G, int TPM, bool CONJ>
__device__ __forceinline__ void cz_middle(double2* trk, int tm, const CzTw<G, TPM>& tw, const double2* __restrict__ hf)
{
    constexpr int R1 = G::R1, R2 = G::R2, R3 = G::R3, L = G::L;
    using T = CzTw<G, TPM>;
#pragma unroll
    for (int i = 0; i < T::NIB; ++i) {
        const int wq = tm + i * TPM;
        if (wq >= L / R2) break;
        const int k1 = wq & (R1 - 1), n2p = wq >> G::LR1;
        double2* base = trk + k1 + G::S3 * n2p;
        double2 u[R2];
#pragma unroll
        for (int t = 0; t < R2; ++t) u[t] = base[G::S2 * t];
        dft<R2, false>(u);
        mul_powers<R2>(u, tw.b[i]);
#pragma unroll
        for (int t = 0; t < R2; ++t) base[G::S2 * t] = u[t];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < T::NIC; ++i) {
        const int wq = tm + i * TPM;
        if (wq >= L / R3) break;
        const int k1 = wq & (R1 - 1), k1p = wq >> G::LR1;
        double2* base = trk + k1 + G::S2 * k1p;
        double2 u[R3];
#pragma unroll
        for (int t = 0; t < R3; ++t) u[t] = base[G::S3 * t];
        dft<R3, false>(u);
        const double2* __restrict__ hb = hf + k1 + R1 * k1p;             // spectrum bin k1 + R1 k1' + R1 R2 t
#pragma unroll
        for (int t = 0; t < R3; ++t) {
            double2 h = __ldg(hb + R1 * R2 * t);
            if (CONJ) h.y = -h.y;
            u[t] = cmul(u[t], h);
        }
        dft<R3, true>(u);
        mul_powers<R3>(u, make_double2(tw.c[i].x, -tw.c[i].y));
#pragma unroll
        for (int t = 0; t < R3; ++t) base[G::S3 * t] = u[t];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < T::NIB; ++i) {
        const int wq = tm + i * TPM;
        if (wq >= L / R2) break;
        const int k1 = wq & (R1 - 1), n2p = wq >> G::LR1;
        double2* base = trk + k1 + G::S3 * n2p;
        double2 u[R2];
#pragma unroll
        for (int t = 0; t < R2; ++t) u[t] = base[G::S2 * t];
        dft<R2, true>(u);
#pragma unroll
        for (int t = 0; t < R2; ++t) base[G::S2 * t] = u[t];
    }
    __syncthreads();
}

}  // namespace p2

// analysis of the cap ring pairs listed in `ring_list` (all with chirp-z length G::L)
// shared memory: [KT transform buffers of LPAD][KT row / bin buffers of NB][mbarrier]; the transform buffers are idle
// during the FFT mapping (the bins sit in the row buffers by then) and serve as the output staging of the TMA stores
template <class G, int KT, int NTH>
__global__ void __launch_bounds__(NTH, 1)
k_ring_analysis_cz(const __grid_constant__ CUtensorMap tmF, DevicePlan d, const int* __restrict__ ring_list, int nrings,
                   const double* __restrict__ maps, int k0, int kmaps, const double2* __restrict__ twL, int planes)
{
    using namespace p2;
    constexpr int R1 = G::R1, R2 = G::R2, R3 = G::R3, L = G::L;
    constexpr int TPM = NTH / KT, MB = NTH / KT;
    constexpr int NB = L / 2 + 8;                         // double2 per map of the row / bin buffer (N <= L / 2 + 1)
    constexpr int SLOT = MB * 2 * KT;
    constexpr int NSLOTS = (KT * G::LPAD) / SLOT >= 8 ? 8 : (KT * G::LPAD) / SLOT;
    constexpr int U = NSLOTS >= 6 ? 3 : NSLOTS >= 4 ? 2 : 1;      // boxes per round; two rounds never share a slot
    static_assert(NSLOTS >= 2 && 2 * U <= NSLOTS && MB <= 256, "output staging");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* tr = reinterpret_cast<double2*>(smem_raw);
    double2* rb = tr + KT * G::LPAD;
    double2* const ostage = tr;
    uint64_t* full = reinterpret_cast<uint64_t*>(rb + KT * NB);

    const int tid = threadIdx.x;
    const int nkp = (kmaps + KT - 1) / KT;
    const long long nitems = (long long)nrings * d.ncomp * nkp;
    const int out_hs = planes ? MB : 1, out_ms = planes ? 1 : 2;
    const double dsig = 4.0 * 3.14159265358979323846 / (double)d.npix;
    if (tid == 0) {
        mbar_init(full, 1);
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();
    auto item_of = [&](long long it, int& p, int& comp, int& kfirst) {
        const int kp = (int)(it % nkp);
        const long long r = it / nkp;
        comp = (int)(r % d.ncomp);
        p = ring_list[(int)(r / d.ncomp)];
        kfirst = kp * KT;
    };
    auto issue_loads = [&](long long it) {
        int p, comp, kfirst;
        item_of(it, p, comp, kfirst);
        const RingPair& rp = d.rings[p];
        const int N = rp.n;
        mbar_arrive_expect_tx(full, (uint32_t)(KT * 2 * N * 8));
#pragma unroll
        for (int kk = 0; kk < KT; ++kk) {
            const int k = min(kfirst + kk, kmaps - 1);
            const double* mp = maps + ((size_t)(k0 + k) * d.ncomp + comp) * d.npix;
            double* dst = reinterpret_cast<double*>(rb + kk * NB);
            bulk_load(dst, mp + rp.start_n, N * 8, full);
            bulk_load(dst + N, mp + rp.start_s, N * 8, full);
        }
    };
    if (tid == 0 && (long long)blockIdx.x < nitems) issue_loads(blockIdx.x);

    const int kkp = tid / TPM, tm = tid - kkp * TPM;
    const int kkm = tid & (KT - 1), mi = tid / KT;
    CzTw<G, TPM> tw;
    tw.load(twL, tm);
    int li = 0, nstore = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x, ++li) {
        int p, comp, kfirst;
        item_of(it, p, comp, kfirst);
        const RingPair rp = d.rings[p];
        const int N = rp.n;
        const double2* __restrict__ hf = d.tw + rp.cz_off;          // [L] filter spectrum, then [N] chirp
        const double2* __restrict__ chirp = hf + L;
        const double2* __restrict__ tw2 = d.tw + rp.tw_off;          // W_{2N}^j (phase of the FFT mapping)
        // phase recurrence of the FFT mapping: d sigma W_{2N}^{mi}, step W_{2N}^{MB} (fetched now, used after the passes)
        double2 phc = __ldg(tw2 + mi % (2 * N));
        phc.x *= dsig; phc.y *= dsig;
        const double2 pstep = __ldg(tw2 + MB % (2 * N));
        mbar_wait(full, li & 1);
        if (tid == 0) bulk_wait_read<0>();                // the stores of the previous item have read the transform buffers
        __syncthreads();
        double2* trk = tr + kkp * G::LPAD;
        // ---- pass A: a_n = x_n c_n (zero past N), R1-point transforms over n1 (stride L / R1), twiddle W_L^{n2 k1}
        {
            const double* rows = reinterpret_cast<const double*>(rb + kkp * NB);
#pragma unroll
            for (int i = 0; i < CzTw<G, TPM>::NIA; ++i) {
                const int j = tm + i * TPM;
                if (j >= L / R1) break;
                double2 u[R1];
#pragma unroll
                for (int r = 0; r < R1; ++r) {
                    const int n = j + r * (L / R1);
                    u[r] = make_double2(0.0, 0.0);       // N <= L / 2: the upper half of the inputs is always zero (pruned at compile time)
                    if (r < R1 / 2 && n < N) u[r] = cmul(make_double2(rows[n], rows[N + n]), __ldg(chirp + n));
                }
                dft<R1, false>(u);
                mul_powers<R1>(u, tw.a[i]);
                const int n1p = j / R3, n2p = j - n1p * R3;
                const int B = n1p + R2 * n2p;
                double2* dst = trk + R1 * B + B + n2p;
#pragma unroll
                for (int k = 0; k < R1; ++k) dst[k] = u[k];
            }
        }
        __syncthreads();
        cz_middle<G, TPM, false>(trk, tm, tw, hf);
        // ---- pass A^-1: y_n, n = n1 L / R1 + n2; bins X_n = y_n c_n for n < N go to the row buffer (the rows are consumed)
        {
            double2* bins = rb + kkp * NB;
#pragma unroll
            for (int i = 0; i < CzTw<G, TPM>::NIA; ++i) {
                const int j = tm + i * TPM;
                if (j >= L / R1) break;
                const int n1p = j / R3, n2p = j - n1p * R3;
                const int B = n1p + R2 * n2p;
                const double2* src = trk + R1 * B + B + n2p;
                double2 u[R1];
#pragma unroll
                for (int q = 0; q < R1; ++q) u[q] = src[q];
                mul_powers<R1>(u, make_double2(tw.a[i].x, -tw.a[i].y));
                dft<R1, true>(u);
#pragma unroll
                for (int r = 0; r < R1 / 2; ++r) {        // outputs n >= L / 2 >= N are never needed
                    const int n = j + r * (L / R1);
                    if (n < N) bins[n] = cmul(u[r], __ldg(chirp + n));
                }
            }
        }
        __syncthreads();
        // ---- FFT mapping from the natural-order bins
        const int mlim = rp.mlim;
        const double2* bm = rb + kkm * NB;
        const int kg = kfirst / KG, csel = (kfirst % KG) / KT;
        for (int m0 = 0; m0 < mlim; m0 += U * MB) {
#pragma unroll
            for (int q = 0; q < U; ++q) {
                const int m = m0 + q * MB + mi;
                const int b = m < N ? m : m % N;
                const int bc = b == 0 ? 0 : N - b;
                const double2 A = bm[b], Bv = bm[bc];
                const double2 gn = make_double2(0.5 * (A.x + Bv.x), 0.5 * (A.y - Bv.y));
                const double2 gs = make_double2(0.5 * (A.y + Bv.y), -0.5 * (A.x - Bv.x));
                const double2 ph = phc;                   // cap rings are all shifted: phi0 = pi / N
                phc = cmul(phc, pstep);
                double2 E = cmul(ph, cadd(gn, gs)), O = cmul(ph, csub(gn, gs));
                if (comp == 1) { E = make_double2(-E.y, E.x); O = make_double2(-O.y, O.x); }
                double2* slot = ostage + ((nstore + q) % NSLOTS) * SLOT;
                slot[(mi * out_ms) * KT + kkm] = E;
                slot[(out_hs + mi * out_ms) * KT + kkm] = O;
            }
            fence_async_smem();
            if (tid == 0) bulk_wait_read<0>();
            __syncthreads();
            if (tid == 0) {
#pragma unroll
                for (int q = 0; q < U; ++q) {
                    const int mq = m0 + q * MB;
                    if (mq >= mlim) break;
                    const double2* slot = ostage + ((nstore + q) % NSLOTS) * SLOT;
                    if (planes) tma_store_5d(&tmF, slot, 0, mq, 2 * comp, csel, p * d.nkg + kg);
                    else tma_store_5d(&tmF, slot, 0, csel, 2 * comp, mq, p * d.nkg + kg);
                }
                bulk_commit();
            }
            nstore += U;
        }
        if (tid == 0 && it + gridDim.x < nitems) issue_loads(it + gridDim.x);
    }
    if (tid == 0) bulk_wait<0>();
}

// synthesis of the cap ring pairs listed in `ring_list` by the chirp-z transform:
//   x_n = conj(c_n) sum_b (Z_b conj(c_b)) c_{n-b}: the same convolution with the conjugated chirp and filter spectrum.
// shared memory: [NSL input slots][KT transform buffers of LPAD][mbarriers].  The ring spectrum is accumulated in the
// transform buffers themselves (natural order, first N elements); every thread owns at most one pass-A butterfly, reads
// its inputs into registers, and the pass writes the buffers in place after a barrier.
template <class G, int KT, int NSL, int NTH>
__global__ void __launch_bounds__(NTH, 1)
k_ring_synthesis_cz(const __grid_constant__ CUtensorMap tmF, DevicePlan d, const int* __restrict__ ring_list, int nrings,
                    double* __restrict__ maps, int k0, int kmaps, const double2* __restrict__ twL, int planes)
{
    using namespace p2;
    constexpr int R1 = G::R1, R2 = G::R2, R3 = G::R3, L = G::L;
    constexpr int TPM = NTH / KT, MB = NTH / KT;
    constexpr int SLOT = MB * 2 * KT;
    static_assert(L / R1 <= TPM && MB <= 256, "one pass-A butterfly per thread");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* in_slots = reinterpret_cast<double2*>(smem_raw);
    double2* tr = in_slots + NSL * SLOT;
    uint64_t* full = reinterpret_cast<uint64_t*>(tr + KT * G::LPAD);

    const int tid = threadIdx.x;
    const int nkp = (kmaps + KT - 1) / KT;
    const long long nitems = (long long)nrings * d.ncomp * nkp;
    const int in_hs = planes ? MB : 1, in_ms = planes ? 1 : 2;
    if (tid == 0) {
        for (int s = 0; s < NSL; ++s) mbar_init(full + s, 1);
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();
    auto item_of = [&](long long it, int& p, int& comp, int& kfirst) {
        const int kp = (int)(it % nkp);
        const long long r = it / nkp;
        comp = (int)(r % d.ncomp);
        p = ring_list[(int)(r / d.ncomp)];
        kfirst = kp * KT;
    };
    // producer (thread 0): the flattened (item, chunk) sequence, NSL chunks ahead
    long long pit = blockIdx.x;
    int pm0 = 0, pmlim = 0, pslot = 0, pp = 0, pcomp = 0, pkf = 0;
    auto producer_begin_item = [&]() {
        if (pit < nitems) { item_of(pit, pp, pcomp, pkf); pmlim = d.rings[pp].mlim; pm0 = 0; }
    };
    auto produce_one = [&]() {
        if (pit >= nitems) return;
        mbar_arrive_expect_tx(full + pslot, SLOT * 16);
        const int kg = pkf / KG, csel = (pkf % KG) / KT;
        if (planes) tma_load_5d(in_slots + pslot * SLOT, &tmF, full + pslot, 0, pm0, 2 * pcomp, csel, pp * d.nkg + kg);
        else tma_load_5d(in_slots + pslot * SLOT, &tmF, full + pslot, 0, csel, 2 * pcomp, pm0, pp * d.nkg + kg);
        pslot = pslot + 1 == NSL ? 0 : pslot + 1;
        pm0 += MB;
        if (pm0 >= pmlim) { pit += gridDim.x; producer_begin_item(); }
    };
    if (tid == 0) {
        producer_begin_item();
        for (int s = 0; s < NSL; ++s) produce_one();
    }

    const int kkp = tid / TPM, tm = tid - kkp * TPM;
    const int kkm = tid & (KT - 1), mi = tid / KT;
    CzTw<G, TPM> tw;
    tw.load(twL, tm);
    int cslot = 0; uint32_t cphase = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x) {
        int p, comp, kfirst;
        item_of(it, p, comp, kfirst);
        const RingPair rp = d.rings[p];
        const int N = rp.n;
        const double2* __restrict__ hf = d.tw + rp.cz_off;
        const double2* __restrict__ chirp = hf + L;
        const double2* __restrict__ tw2 = d.tw + rp.tw_off;
        double2 phc = __ldg(tw2 + mi % (2 * N));          // e^{+i m phi0} by recurrence, step W_{2N}^{-MB}
        phc.y = -phc.y;
        double2 pstep = __ldg(tw2 + MB % (2 * N));
        pstep.y = -pstep.y;
        for (int i = tid; i < KT * N; i += NTH) { const int kz = i / N; tr[kz * G::LPAD + (i - kz * N)] = make_double2(0.0, 0.0); }
        __syncthreads();
        // ---- inverse FFT mapping: accumulate the ring spectrum Z_b, b < N (as in the belt kernel)
        const int mlim = rp.mlim;
        double2* zm = tr + kkm * G::LPAD;
        for (int m0 = 0; m0 < mlim; m0 += MB) {
            mbar_wait(full + cslot, cphase);
            const double2* slot = in_slots + cslot * SLOT;
            const int m = m0 + mi;
            const bool live = m < mlim;
            double2 zd = make_double2(0.0, 0.0), zc = zd;
            if (live) {
                const double2 e = slot[(mi * in_ms) * KT + kkm], o = slot[(in_hs + mi * in_ms) * KT + kkm];
                double2 fn = cadd(e, o), fs = csub(e, o);
                if (comp == 1) { fn = make_double2(fn.y, -fn.x); fs = make_double2(fs.y, -fs.x); }
                double2 ph = phc;
                const double wgt = (m == 0) ? 0.5 : 1.0;
                ph.x *= wgt; ph.y *= wgt;
                const double2 dn = cmul(ph, fn), ds = cmul(ph, fs);
                zd = make_double2(dn.x - ds.y, dn.y + ds.x);
                zc = make_double2(dn.x + ds.y, ds.x - dn.y);
            }
            phc = cmul(phc, pstep);
            const int b1 = m < N ? m : m % N, b2 = b1 == 0 ? 0 : N - b1;
            // two orders of one chunk meet in a bin only if m + m' = 0 mod N for some pair of the chunk
            const bool clash = ((2 * m0 + N - 1) / N) * N <= 2 * m0 + 2 * MB - 2;
            if (live) { double2* c1 = zm + b1; *c1 = cadd(*c1, zd); }
            if (clash) __syncthreads();
            if (live) { double2* c2 = zm + b2; *c2 = cadd(*c2, zc); }
            __syncthreads();
            if (tid == 0) produce_one();
            if (++cslot == NSL) { cslot = 0; cphase ^= 1; }
        }
        double2* trk = tr + kkp * G::LPAD;
        // ---- pass A in place: a_b = Z_b conj(c_b) (zero past N) to registers, barrier, transform, write
        {
            const int j = tm;
            const bool act = j < L / R1;
            double2 u[R1];
            if (act) {
#pragma unroll
                for (int r = 0; r < R1; ++r) {
                    const int n = j + r * (L / R1);
                    u[r] = make_double2(0.0, 0.0);       // N <= L / 2: the upper half of the inputs is always zero
                    if (r < R1 / 2 && n < N) { double2 c = __ldg(chirp + n); c.y = -c.y; u[r] = cmul(trk[n], c); }
                }
            }
            __syncthreads();
            if (act) {
                dft<R1, false>(u);
                mul_powers<R1>(u, tw.a[0]);
                const int n1p = j / R3, n2p = j - n1p * R3;
                const int B = n1p + R2 * n2p;
                double2* dst = trk + R1 * B + B + n2p;
#pragma unroll
                for (int k = 0; k < R1; ++k) dst[k] = u[k];
            }
        }
        __syncthreads();
        cz_middle<G, TPM, true>(trk, tm, tw, hf);
        // ---- pass A^-1: pixels x_n = y_n conj(c_n), north = real part, south = imaginary part
        {
            const int k = kfirst + kkp;
            double* mp = maps + ((size_t)(k0 + (k < kmaps ? k : 0)) * d.ncomp + comp) * d.npix;
#pragma unroll
            for (int i = 0; i < CzTw<G, TPM>::NIA; ++i) {
                const int j = tm + i * TPM;
                if (j >= L / R1) break;
                const int n1p = j / R3, n2p = j - n1p * R3;
                const int B = n1p + R2 * n2p;
                const double2* src = trk + R1 * B + B + n2p;
                double2 u[R1];
#pragma unroll
                for (int q = 0; q < R1; ++q) u[q] = src[q];
                mul_powers<R1>(u, make_double2(tw.a[i].x, -tw.a[i].y));
                dft<R1, true>(u);
                if (k < kmaps) {
#pragma unroll
                    for (int r = 0; r < R1 / 2; ++r) {    // pixels n >= L / 2 >= N do not exist
                        const int n = j + r * (L / R1);
                        if (n < N) {
                            double2 c = __ldg(chirp + n); c.y = -c.y;
                            const double2 x = cmul(u[r], c);
                            mp[rp.start_n + n] = x.x;
                            mp[rp.start_s + n] = x.y;
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
}

// ---- host side -------------------------------------------------------------------------------------------
template <int LOGN, int KT, int NSL>
static size_t synthesis_p2_smem()
{
    return (size_t)NSL * (p2::NT / KT) * 2 * KT * 16 + (size_t)KT * p2::buf_stride<LOGN, KT>() * 16 + 8 * NSL + 64;
}

template <int LOGN, int KT>
static cudaError_t run_analysis_p2i(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    const size_t sm = (size_t)KT * p2::buf_stride<LOGN, KT>() * 16 + (size_t)4 * (p2::NT / KT) * 2 * KT * 16 + 64;
    cudaError_t e = cudaFuncSetAttribute(k_ring_analysis_p2i<LOGN, KT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, p2::NT / KT, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, p2::NT / KT, false, &tm)) != cudaSuccess) return e;
    }
    const long long nitems = (long long)pl->belt_count * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = 2LL * pl->sm_count;
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    k_ring_analysis_p2i<LOGN, KT><<<grid, p2::NT, sm, st>>>(tm, d, maps, k0, kmaps, pl->belt_first, pl->belt_count, planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

template <int LOGN, int KT, int NSL>
static cudaError_t run_synthesis_p2(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    const size_t sm = synthesis_p2_smem<LOGN, KT, NSL>();
    cudaError_t e = cudaFuncSetAttribute(k_ring_synthesis_p2<LOGN, KT, NSL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, p2::NT / KT, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, p2::NT / KT, false, &tm)) != cudaSuccess) return e;
    }
    const long long nitems = (long long)pl->belt_count * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = 2LL * pl->sm_count;           // two CTAs per SM
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    k_ring_synthesis_p2<LOGN, KT, NSL><<<grid, p2::NT, sm, st>>>(tm, d, maps, k0, kmaps, pl->belt_first, pl->belt_count, planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

template <class G, int KT>
static cudaError_t run_analysis_cz(sht_plan_s* pl, const DevicePlan& d, int cls, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    constexpr int NTH = 512, MB = NTH / KT;
    const size_t sm = (size_t)KT * G::LPAD * 16 + (size_t)KT * (G::L / 2 + 8) * 16 + 64;
    auto kern = k_ring_analysis_cz<G, KT, NTH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, MB, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, MB, false, &tm)) != cudaSuccess) return e;
    }
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, NTH, sm) != cudaSuccess || occ < 1) { cudaGetLastError(); occ = 1; }
    const long long nitems = (long long)pl->cz_count[cls] * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = (long long)pl->sm_count * occ;
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    kern<<<grid, NTH, sm, st>>>(tm, d, pl->cz_rings[cls], pl->cz_count[cls], maps, k0, kmaps, d.tw + pl->cz_tw_off[cls], planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

template <class G, int KT>
static cudaError_t run_synthesis_cz(sht_plan_s* pl, const DevicePlan& d, int cls, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    constexpr int NTH = 512, MB = NTH / KT, NSL = 2;
    const size_t sm = (size_t)KT * G::LPAD * 16 + (size_t)NSL * MB * 2 * KT * 16 + 64;
    auto kern = k_ring_synthesis_cz<G, KT, NSL, NTH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, MB, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, MB, false, &tm)) != cudaSuccess) return e;
    }
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, NTH, sm) != cudaSuccess || occ < 1) { cudaGetLastError(); occ = 1; }
    const long long nitems = (long long)pl->cz_count[cls] * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = (long long)pl->sm_count * occ;
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    kern<<<grid, NTH, sm, st>>>(tm, d, pl->cz_rings[cls], pl->cz_count[cls], maps, k0, kmaps, d.tw + pl->cz_tw_off[cls], planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

// cap rings on the chirp-z path: one persistent launch per compiled convolution length, longest first
cudaError_t launch_ring_analysis_cz(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    using namespace p2;
    cudaError_t e = cudaSuccess;
    for (int c = CZ_NCLASS - 1; c >= 0 && e == cudaSuccess; --c) {
        if (pl->cz_count[c] == 0) continue;
        switch (CZ_LEN[c]) {
            case 512: e = run_analysis_cz<GeoT<8, 8, 8>, 4>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 768: e = run_analysis_cz<GeoT<8, 8, 12>, 4>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 1024: e = run_analysis_cz<GeoT<16, 8, 8>, 4>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 1536: e = run_analysis_cz<GeoT<16, 8, 12>, 2>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 2048: e = run_analysis_cz<GeoT<16, 16, 8>, 2>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 3072: e = run_analysis_cz<GeoT<16, 16, 12>, 2>(pl, d, c, maps, F, k0, kmaps, st); break;
            case 4096: e = run_analysis_cz<GeoT<16, 16, 16>, 2>(pl, d, c, maps, F, k0, kmaps, st); break;
            default: e = cudaErrorNotSupported;
        }
    }
    return e;
}

cudaError_t launch_ring_synthesis_cz(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    using namespace p2;
    cudaError_t e = cudaSuccess;
    for (int c = CZ_NCLASS - 1; c >= 0 && e == cudaSuccess; --c) {
        if (pl->cz_count[c] == 0) continue;
        switch (CZ_LEN[c]) {
            case 512: e = run_synthesis_cz<GeoT<8, 8, 8>, 4>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 768: e = run_synthesis_cz<GeoT<8, 8, 12>, 4>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 1024: e = run_synthesis_cz<GeoT<16, 8, 8>, 4>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 1536: e = run_synthesis_cz<GeoT<16, 8, 12>, 2>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 2048: e = run_synthesis_cz<GeoT<16, 16, 8>, 2>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 3072: e = run_synthesis_cz<GeoT<16, 16, 12>, 2>(pl, d, c, F, maps, k0, kmaps, st); break;
            case 4096: e = run_synthesis_cz<GeoT<16, 16, 16>, 2>(pl, d, c, F, maps, k0, kmaps, st); break;
            default: e = cudaErrorNotSupported;
        }
    }
    return e;
}

// belt ring pairs of a power-of-two nside through the fast path; returns cudaErrorNotSupported if this plan has none
cudaError_t launch_ring_analysis_belt(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    switch (pl->belt_logn) {
        case 9: return run_analysis_p2i<9, 4>(pl, d, maps, F, k0, kmaps, st);
        case 10: return run_analysis_p2i<10, 4>(pl, d, maps, F, k0, kmaps, st);
        case 11: return run_analysis_p2i<11, 2>(pl, d, maps, F, k0, kmaps, st);
        default: return cudaErrorNotSupported;
    }
}

cudaError_t launch_ring_synthesis_belt(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    switch (pl->belt_logn) {
        case 9: return run_synthesis_p2<9, 4, 4>(pl, d, F, maps, k0, kmaps, st);
        case 10: return run_synthesis_p2<10, 4, 4>(pl, d, F, maps, k0, kmaps, st);
        case 11: return run_synthesis_p2<11, 2, 4>(pl, d, F, maps, k0, kmaps, st);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace sht
