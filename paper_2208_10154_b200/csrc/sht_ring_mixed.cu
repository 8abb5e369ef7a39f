// sht_ring_mixed.cu -- subsystem (1), cap rings whose length N = 4 i factors into three radices with prime factors
// <= 31: a direct mixed-radix transform N = R1 R2 R3 (PAPER.md:47-54 eq. 2 row 3; :66-70 eq. 4), three passes in
// registers with the codelets of sht_dft_codelets.cuh.  Same structure as the belt kernels of sht_ring_pow2.cu
// (decimation in time on the analysis side: first pass from the bulk-copied rows, bins in natural order for the FFT
// mapping, lines out by TMA stores; the adjoint network on the synthesis side), with the radices and strides of the
// ring read from the plan at run time: a pass dispatches on its own radix only (compile-time codelet), the other two
// radices enter through index arithmetic (one multiply-high per butterfly instead of a division).
// Rings that do not factor this way take the chirp-z path (sht_ring_pow2.cu) or the general kernels.
#include "sht_ring_common.cuh"
#include "sht_dft_codelets.cuh"

namespace sht {

namespace mr {

using p2::cmul; using p2::cadd; using p2::csub;
constexpr int NT = 256;

// position of element p in a transform buffer: one element of padding per 16
__device__ __forceinline__ int phys(int p) { return p + (p >> 4); }
// (a multiple of 8 elements, so that what follows the transform buffers stays 128-byte aligned for the TMA engine)
__host__ __device__ constexpr int padded(int n) { return (n + n / 16 + 8 + 7) & ~7; }
// floor(x / d) for x < 2^16 by a multiply-high with mg = floor((2^32 - 1) / d) + 1
__device__ __forceinline__ int divm(int x, unsigned mg) { return (int)__umulhi((unsigned)x, mg); }

struct Radices {
    int r1, r2, r3;
    unsigned mg1, mg3;                                   // magic numbers of the divisions by r1 and r3
};

// ---- forward passes --------------------------------------------------------------------------------------
// pass A: R1-point transforms over n1 (input stride N / R1) from the staged rows, twiddle W_N^{n2 k1}, written to R1
// consecutive positions R1 (n1' + R2 n2') + k1, where n2 = R3 n1' + n2'
template <int R>
__device__ __forceinline__ void fwd_a(const double* rows, int N, double2* trk, int tm, int tpm, const Radices& q,
                                      const double2* __restrict__ tw2)
{
    const int cnt = N / R;
    for (int j = tm; j < cnt; j += tpm) {
        double2 u[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { u[r].x = rows[j + r * cnt]; u[r].y = rows[N + j + r * cnt]; }
        const double2 w = __ldg(tw2 + 2 * j);
        dftc::Dft<R, false>::run(u);
        dftc::mul_powers_any<R>(u, w);
        const int n1p = divm(j, q.mg3), n2p = j - n1p * q.r3;
        const int base = R * (n1p + q.r2 * n2p);
#pragma unroll
        for (int k = 0; k < R; ++k) trk[phys(base + k)] = u[k];
    }
}
// pass B: R2-point transforms over n1' at positions k1 + R1 t + R1 R2 n2', twiddle W_N^{R1 n2' k1'}
template <int R>
__device__ __forceinline__ void fwd_b(int N, double2* trk, int tm, int tpm, const Radices& q, const double2* __restrict__ tw2)
{
    const int cnt = N / R;
    for (int wq = tm; wq < cnt; wq += tpm) {
        const int n2p = divm(wq, q.mg1), k1 = wq - n2p * q.r1;
        const int base = k1 + q.r1 * R * n2p;
        double2 u[R];
#pragma unroll
        for (int t = 0; t < R; ++t) u[t] = trk[phys(base + q.r1 * t)];
        const double2 w = __ldg(tw2 + 2 * q.r1 * n2p);
        dftc::Dft<R, false>::run(u);
        dftc::mul_powers_any<R>(u, w);
#pragma unroll
        for (int t = 0; t < R; ++t) trk[phys(base + q.r1 * t)] = u[t];
    }
}
// pass C: R3-point transforms over n2' at positions k1 + R1 k1' + R1 R2 t; bin k1 + R1 k1' + R1 R2 k2' in place
template <int R, bool INV>
__device__ __forceinline__ void pass_c(int N, double2* trk, int tm, int tpm, const Radices& q, const double2* __restrict__ tw2)
{
    const int cnt = N / R, s3 = q.r1 * q.r2;
    for (int wq = tm; wq < cnt; wq += tpm) {
        const int k1p = divm(wq, q.mg1), k1 = wq - k1p * q.r1;
        const int base = k1 + q.r1 * k1p;
        double2 u[R];
#pragma unroll
        for (int t = 0; t < R; ++t) u[t] = trk[phys(base + s3 * t)];
        dftc::Dft<R, INV>::run(u);
        if (INV) {                                        // adjoint network: conjugate twiddle W_N^{-R1 k1' n2'}
            double2 w = __ldg(tw2 + 2 * q.r1 * k1p);
            w.y = -w.y;
            dftc::mul_powers_any<R>(u, w);
        }
#pragma unroll
        for (int t = 0; t < R; ++t) trk[phys(base + s3 * t)] = u[t];
    }
}
// pass B^-1: inverse R2-point transforms over k1'
template <int R>
__device__ __forceinline__ void inv_b(int N, double2* trk, int tm, int tpm, const Radices& q)
{
    const int cnt = N / R;
    for (int wq = tm; wq < cnt; wq += tpm) {
        const int n2p = divm(wq, q.mg1), k1 = wq - n2p * q.r1;
        const int base = k1 + q.r1 * R * n2p;
        double2 u[R];
#pragma unroll
        for (int t = 0; t < R; ++t) u[t] = trk[phys(base + q.r1 * t)];
        dftc::Dft<R, true>::run(u);
#pragma unroll
        for (int t = 0; t < R; ++t) trk[phys(base + q.r1 * t)] = u[t];
    }
}
// pass A^-1: conjugate twiddle W_N^{-n2 k1}, inverse R1-point transforms over k1 -> pixels n1 N / R1 + n2 of the two rings
template <int R>
__device__ __forceinline__ void inv_a(int N, const double2* trk, int tm, int tpm, const Radices& q, const double2* __restrict__ tw2,
                                      double* north, double* south, bool write)
{
    const int cnt = N / R;
    for (int j = tm; j < cnt; j += tpm) {
        const int n1p = divm(j, q.mg3), n2p = j - n1p * q.r3;
        const int base = R * (n1p + q.r2 * n2p);
        double2 u[R];
#pragma unroll
        for (int k = 0; k < R; ++k) u[k] = trk[phys(base + k)];
        double2 w = __ldg(tw2 + 2 * j);
        w.y = -w.y;
        dftc::mul_powers_any<R>(u, w);
        dftc::Dft<R, true>::run(u);
        if (write) {
#pragma unroll
            for (int r = 0; r < R; ++r) { north[j + r * cnt] = u[r].x; south[j + r * cnt] = u[r].y; }
        }
    }
}

// the radices a plan may hand out (sht_plan.cu picks three of them per ring length); kernels compiled with BIG = false
// know the radices up to 16 only and fit two CTAs per SM, the others also take 17 .. 31 (one CTA per SM)
#define SHT_MR_DISPATCH(R, CALL)                                                                                      \
    switch (R) {                                                                                                      \
        case 2: CALL(2); break; case 3: CALL(3); break; case 4: CALL(4); break; case 5: CALL(5); break;              \
        case 6: CALL(6); break; case 7: CALL(7); break; case 8: CALL(8); break; case 9: CALL(9); break;              \
        case 10: CALL(10); break; case 11: CALL(11); break; case 12: CALL(12); break; case 13: CALL(13); break;      \
        case 14: CALL(14); break; case 15: CALL(15); break; case 16: CALL(16); break;                                \
        default:                                                                                                      \
            if constexpr (BIG) {                                                                                      \
                switch (R) {                                                                                          \
                    case 17: CALL(17); break; case 19: CALL(19); break; case 20: CALL(20); break;                     \
                    case 23: CALL(23); break; case 29: CALL(29); break; case 31: CALL(31); break; default: break;    \
                }                                                                                                     \
            }                                                                                                         \
            break;                                                                                                    \
    }

}  // namespace mr

// ------------------------------------------------------------------------------------------------
// analysis of the cap ring pairs in `ring_list` (mixed-radix path); KT maps per item, 256 threads
// shared memory: [KT row buffers of 2 nmax doubles][KT transform buffers of padded(nmax)][4 output slots][mbarrier]
// ------------------------------------------------------------------------------------------------
template <int KT, bool BIG>
__global__ void __launch_bounds__(mr::NT, BIG ? 1 : 2)
k_ring_analysis_mr(const __grid_constant__ CUtensorMap tmF, DevicePlan d, const int* __restrict__ ring_list, int nrings, int nmax,
                   const double* __restrict__ maps, int k0, int kmaps, int planes)
{
    using namespace mr;
    using namespace p2;
    constexpr int TPM = mr::NT / KT, MB = mr::NT / KT, SLOT = MB * 2 * KT, NSLOTS = 4, U = 2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* rowsb = reinterpret_cast<double*>(smem_raw);
    double2* tr = reinterpret_cast<double2*>(rowsb + (size_t)KT * 2 * nmax);
    const int np = padded(nmax);
    double2* ostage = tr + (size_t)KT * np;
    uint64_t* full = reinterpret_cast<uint64_t*>(ostage + NSLOTS * SLOT);

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
            double* dst = rowsb + (size_t)kk * 2 * nmax;
            bulk_load(dst, mp + rp.start_n, N * 8, full);
            bulk_load(dst + N, mp + rp.start_s, N * 8, full);
        }
    };
    if (tid == 0 && (long long)blockIdx.x < nitems) issue_loads(blockIdx.x);

    const int kkp = tid / TPM, tm = tid - kkp * TPM;
    const int kkm = tid & (KT - 1), mi = tid / KT;
    int li = 0, nstore = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x, ++li) {
        int p, comp, kfirst;
        item_of(it, p, comp, kfirst);
        const RingPair rp = d.rings[p];
        const int N = rp.n;
        const double2* __restrict__ tw2 = d.tw + rp.tw_off;          // W_{2N}^j; W_N^e = tw2[2 e]
        Radices q;
        q.r1 = rp.mr_r1; q.r2 = rp.mr_r2; q.r3 = rp.mr_r3;
        q.mg1 = 0xFFFFFFFFu / (unsigned)q.r1 + 1u; q.mg3 = 0xFFFFFFFFu / (unsigned)q.r3 + 1u;
        // phase recurrence of the FFT mapping: d sigma W_{2N}^{mi}, step W_{2N}^{MB}
        double2 phc = __ldg(tw2 + mi % (2 * N));
        phc.x *= dsig; phc.y *= dsig;
        const double2 pstep = __ldg(tw2 + MB % (2 * N));
        mbar_wait(full, li & 1);
        const double* rows = rowsb + (size_t)kkp * 2 * nmax;
        double2* trk = tr + (size_t)kkp * np;
#define SHT_CALL(R) fwd_a<R>(rows, N, trk, tm, TPM, q, tw2)
        SHT_MR_DISPATCH(q.r1, SHT_CALL)
#undef SHT_CALL
        __syncthreads();
        // the row buffers are free: fetch the next item's rows while this one is transformed
        if (tid == 0 && it + gridDim.x < nitems) issue_loads(it + gridDim.x);
#define SHT_CALL(R) fwd_b<R>(N, trk, tm, TPM, q, tw2)
        SHT_MR_DISPATCH(q.r2, SHT_CALL)
#undef SHT_CALL
        __syncthreads();
        if (q.r3 > 1) {
#define SHT_CALL(R) pass_c<R, false>(N, trk, tm, TPM, q, tw2)
            SHT_MR_DISPATCH(q.r3, SHT_CALL)
#undef SHT_CALL
            __syncthreads();
        }
        // ---- FFT mapping from the natural-order bins
        const int mlim = rp.mlim;
        const double2* bm = tr + (size_t)kkm * np;
        const int kg = kfirst / KG, csel = (kfirst % KG) / KT;
        for (int m0 = 0; m0 < mlim; m0 += U * MB) {
#pragma unroll
            for (int u_ = 0; u_ < U; ++u_) {
                const int m = m0 + u_ * MB + mi;
                const int b = m < N ? m : m % N;
                const int bc = b == 0 ? 0 : N - b;
                const double2 A = bm[phys(b)], Bv = bm[phys(bc)];
                const double2 gn = make_double2(0.5 * (A.x + Bv.x), 0.5 * (A.y - Bv.y));
                const double2 gs = make_double2(0.5 * (A.y + Bv.y), -0.5 * (A.x - Bv.x));
                const double2 ph = phc;                   // cap rings are all shifted: phi0 = pi / N
                phc = cmul(phc, pstep);
                double2 E = cmul(ph, cadd(gn, gs)), O = cmul(ph, csub(gn, gs));
                if (comp == 1) { E = make_double2(-E.y, E.x); O = make_double2(-O.y, O.x); }
                double2* slot = ostage + ((nstore + u_) % NSLOTS) * SLOT;
                slot[(mi * out_ms) * KT + kkm] = E;
                slot[(out_hs + mi * out_ms) * KT + kkm] = O;
            }
            fence_async_smem();
            if (tid == 0) bulk_wait_read<0>();
            __syncthreads();
            if (tid == 0) {
#pragma unroll
                for (int u_ = 0; u_ < U; ++u_) {
                    const int mq = m0 + u_ * MB;
                    if (mq >= mlim) break;
                    const double2* slot = ostage + ((nstore + u_) % NSLOTS) * SLOT;
                    if (planes) tma_store_5d(&tmF, slot, 0, mq, 2 * comp, csel, p * d.nkg + kg);
                    else tma_store_5d(&tmF, slot, 0, csel, 2 * comp, mq, p * d.nkg + kg);
                }
                bulk_commit();
            }
            nstore += U;
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// ------------------------------------------------------------------------------------------------
// synthesis of the cap ring pairs in `ring_list` (mixed-radix path)
// shared memory: [NSL input slots][KT transform buffers of padded(nmax)][mbarriers]
// ------------------------------------------------------------------------------------------------
template <int KT, int NSL, bool BIG>
__global__ void __launch_bounds__(mr::NT, BIG ? 1 : 2)
k_ring_synthesis_mr(const __grid_constant__ CUtensorMap tmF, DevicePlan d, const int* __restrict__ ring_list, int nrings, int nmax,
                    double* __restrict__ maps, int k0, int kmaps, int planes)
{
    using namespace mr;
    using namespace p2;
    constexpr int TPM = mr::NT / KT, MB = mr::NT / KT, SLOT = MB * 2 * KT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* in_slots = reinterpret_cast<double2*>(smem_raw);
    double2* tr = in_slots + NSL * SLOT;
    const int np = padded(nmax);
    uint64_t* full = reinterpret_cast<uint64_t*>(tr + (size_t)KT * np);

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
    int cslot = 0; uint32_t cphase = 0;
    for (long long it = blockIdx.x; it < nitems; it += gridDim.x) {
        int p, comp, kfirst;
        item_of(it, p, comp, kfirst);
        const RingPair rp = d.rings[p];
        const int N = rp.n;
        const double2* __restrict__ tw2 = d.tw + rp.tw_off;
        Radices q;
        q.r1 = rp.mr_r1; q.r2 = rp.mr_r2; q.r3 = rp.mr_r3;
        q.mg1 = 0xFFFFFFFFu / (unsigned)q.r1 + 1u; q.mg3 = 0xFFFFFFFFu / (unsigned)q.r3 + 1u;
        double2 phc = __ldg(tw2 + mi % (2 * N));          // e^{+i m phi0} by recurrence
        phc.y = -phc.y;
        double2 pstep = __ldg(tw2 + MB % (2 * N));
        pstep.y = -pstep.y;
        const int npn = padded(N);
        for (int i = tid; i < KT * npn; i += mr::NT) { const int kz = i / npn; tr[(size_t)kz * np + (i - kz * npn)] = make_double2(0.0, 0.0); }
        __syncthreads();
        // ---- inverse FFT mapping: accumulate the ring spectrum Z_b (as in the belt kernel)
        const int mlim = rp.mlim;
        double2* zm = tr + (size_t)kkm * np;
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
            const bool clash = ((2 * m0 + N - 1) / N) * N <= 2 * m0 + 2 * MB - 2;
            if (live) { double2* c1 = zm + phys(b1); *c1 = cadd(*c1, zd); }
            if (clash) __syncthreads();
            if (live) { double2* c2 = zm + phys(b2); *c2 = cadd(*c2, zc); }
            __syncthreads();
            if (tid == 0) produce_one();
            if (++cslot == NSL) { cslot = 0; cphase ^= 1; }
        }
        double2* trk = tr + (size_t)kkp * np;
        if (q.r3 > 1) {
#define SHT_CALL(R) pass_c<R, true>(N, trk, tm, TPM, q, tw2)
            SHT_MR_DISPATCH(q.r3, SHT_CALL)
#undef SHT_CALL
            __syncthreads();
        }
#define SHT_CALL(R) inv_b<R>(N, trk, tm, TPM, q)
        SHT_MR_DISPATCH(q.r2, SHT_CALL)
#undef SHT_CALL
        __syncthreads();
        const int k = kfirst + kkp;
        double* mp = maps + ((size_t)(k0 + (k < kmaps ? k : 0)) * d.ncomp + comp) * d.npix;
#define SHT_CALL(R) inv_a<R>(N, trk, tm, TPM, q, tw2, mp + rp.start_n, mp + rp.start_s, k < kmaps)
        SHT_MR_DISPATCH(q.r1, SHT_CALL)
#undef SHT_CALL
        __syncthreads();
    }
}

// ---- host side -------------------------------------------------------------------------------------------
template <int KT, bool BIG>
static cudaError_t run_analysis_mr(sht_plan_s* pl, const DevicePlan& d, int cls, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    constexpr int MB = mr::NT / KT;
    const int nmax = pl->mr_nmax[cls];
    const size_t sm = (size_t)KT * 2 * nmax * 8 + (size_t)KT * mr::padded(nmax) * 16 + (size_t)4 * MB * 2 * KT * 16 + 64;
    auto kern = k_ring_analysis_mr<KT, BIG>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, MB, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, MB, false, &tm)) != cudaSuccess) return e;
    }
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, mr::NT, sm) != cudaSuccess || occ < 1) { cudaGetLastError(); occ = 1; }
    const long long nitems = (long long)pl->mr_count[cls] * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = (long long)pl->sm_count * occ;
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    kern<<<grid, mr::NT, sm, st>>>(tm, d, pl->mr_rings[cls], pl->mr_count[cls], nmax, maps, k0, kmaps, planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

template <int KT, bool BIG>
static cudaError_t run_synthesis_mr(sht_plan_s* pl, const DevicePlan& d, int cls, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    constexpr int MB = mr::NT / KT, NSL = 4;
    const int nmax = pl->mr_nmax[cls];
    const size_t sm = (size_t)NSL * MB * 2 * KT * 16 + (size_t)KT * mr::padded(nmax) * 16 + 64;
    auto kern = k_ring_synthesis_mr<KT, NSL, BIG>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    bool planes = true;
    if (make_tmap_ring(d, F, KT, MB, true, &tm) != cudaSuccess) {
        planes = false;
        if ((e = make_tmap_ring(d, F, KT, MB, false, &tm)) != cudaSuccess) return e;
    }
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, mr::NT, sm) != cudaSuccess || occ < 1) { cudaGetLastError(); occ = 1; }
    const long long nitems = (long long)pl->mr_count[cls] * d.ncomp * ((kmaps + KT - 1) / KT);
    const long long want = (long long)pl->sm_count * occ;
    const unsigned grid = (unsigned)(nitems < want ? nitems : want);
    kern<<<grid, mr::NT, sm, st>>>(tm, d, pl->mr_rings[cls], pl->mr_count[cls], nmax, maps, k0, kmaps, planes ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

// classes: length class 0: N <= 512 (4 maps per item), 1: N <= 1024 (4 maps), 2: N <= 2048 (2 maps), + 3 if a radix
// above 16 occurs; longest first
cudaError_t launch_ring_analysis_mr(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    for (int c = 2 * MR_NCLASS - 1; c >= 0 && e == cudaSuccess; --c) {
        if (pl->mr_count[c] == 0) continue;
        const bool big = c >= MR_NCLASS, two = (c % MR_NCLASS) == 2;
        e = big ? (two ? run_analysis_mr<2, true>(pl, d, c, maps, F, k0, kmaps, st) : run_analysis_mr<4, true>(pl, d, c, maps, F, k0, kmaps, st))
                : (two ? run_analysis_mr<2, false>(pl, d, c, maps, F, k0, kmaps, st) : run_analysis_mr<4, false>(pl, d, c, maps, F, k0, kmaps, st));
    }
    return e;
}

cudaError_t launch_ring_synthesis_mr(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st)
{
    cudaError_t e = cudaSuccess;
    for (int c = 2 * MR_NCLASS - 1; c >= 0 && e == cudaSuccess; --c) {
        if (pl->mr_count[c] == 0) continue;
        const bool big = c >= MR_NCLASS, two = (c % MR_NCLASS) == 2;
        e = big ? (two ? run_synthesis_mr<2, true>(pl, d, c, F, maps, k0, kmaps, st) : run_synthesis_mr<4, true>(pl, d, c, F, maps, k0, kmaps, st))
                : (two ? run_synthesis_mr<2, false>(pl, d, c, F, maps, k0, kmaps, st) : run_synthesis_mr<4, false>(pl, d, c, F, maps, k0, kmaps, st));
    }
    return e;
}

}  // namespace sht
