// sht_legendre_spin2.cu -- subsystem (2) for spin 2: fused lambda recurrence -> F+/F- (App. A.2)
// -> FP64 tensor-core contraction of the 2 x 2 block products of eq. 14 / eq. 15, and subsystem (3): the E/B
// combination a_E = A^E, a_B = -i (iA^B) (eq. 10) in the epilogue / operand fetch.
//
//   analysis  (eq. 14):  (A^E; iA^B)_m = [[F+, F-], [F-, F+]]_m (Q; iU)_m      contraction over ring pairs
//   synthesis (eq. 15):  (Q; iU)_m = [[F+, F-], [F-, F+]]_m^t (A^E; iA^B)_m    contraction over l
// with F+ = -X1, F- = -X2 (eq. A5; reading G12),
//   X1_lm = N_l { -[(l - m^2)/s^2 + l(l-1)/2] lambda_lm + (x/s^2) c_lm lambda_{l-1,m} }
//   X2_lm = N_l (m/s^2) { c_lm lambda_{l-1,m} - (l-1) x lambda_lm },
//   N_l = 2/sqrt((l-1) l (l+1)(l+2)), c_lm = sqrt((2l+1)/(2l-1) (l^2 - m^2)), x = cos(theta), s = sin(theta).
// Under theta -> pi - theta F+ has the parity (-1)^(l+m) of lambda and F- the opposite one, so for l - m even F+
// meets the E-folded (north + south) and F- the O-folded (north - south) ring coefficients, and vice versa for
// l - m odd.  One pass over the Q and iU tiles of a stage feeds both outputs (item 12).
//
// Same warp-specialised structure as the spin-0 kernels: 8 DMMA consumer warps (CTA tile 128 x 128 real outputs), but
// the four remaining warps all generate (lane = ring x sign of F), and lane 0 of the generator that owns a stage
// also issues its TMA loads.
#include <type_traits>
#include "sht_legendre_common.cuh"

namespace sht {

constexpr int LEG2_THREADS = 384;
constexpr int LEG_CONSUMER_WARPS_S2 = 8;
constexpr int P_KT = 32;                        // (Q,U) pairs per k-tile: 32 pairs x (E,B) x (re,im) = 128 real columns
constexpr int P_KG = P_KT / KG;                 // workspace map groups per k-tile
constexpr int A2_ML = LEG_A_ML;                 // analysis: l rows per tile (64 of each parity class)
constexpr int A2_PC = 16;                       // analysis: ring pairs per stage
constexpr int A2_SL = 66;                       // F tile: stride (doubles) between rings, = 2 mod 8
constexpr int A2_XBYTES = A2_PC * P_KG * 2 * 128;           // Q and iU lines of a stage: 32 KB
constexpr int A2_LBYTES = 2 * 2 * A2_PC * A2_SL * 8;        // [sign][class][ring][l/2]
constexpr int A2_STAGE_BYTES = A2_XBYTES + A2_LBYTES;
static_assert(A2_STAGE_BYTES % 1024 == 0, "stages must keep the 1024-byte alignment of the swizzled TMA boxes");
constexpr int S2_PB = 64;                       // synthesis: ring pairs per CTA
constexpr int S2_LC = 32;                       // synthesis: l values per stage
constexpr int S2_SL = 66;
constexpr int S2_ABYTES = S2_LC * 2 * P_KT * 16;            // a_E, a_B of a stage: 32 KB
constexpr int S2_LBYTES = 2 * S2_LC * S2_SL * 8;            // [sign][l][ring]
constexpr int S2_STAGE_BYTES = S2_ABYTES + S2_LBYTES;
static_assert(S2_STAGE_BYTES % 1024 == 0, "stages must keep the 1024-byte alignment of the swizzled TMA boxes");

// per-l constants of F+/F- for order m: tp = (t1, t2) = N_l (l - m^2, l(l-1)/2), tm = (t4, 0) = N_l (l-1, 0),
// t3 = N_l c_lm; all zero for l < 2 (reading G13) and beyond lmax
__device__ __forceinline__ void spin2_consts(const DevicePlan& d, int l, int m, double2& tp, double2& tm, double& t3)
{
    tp = make_double2(0.0, 0.0); tm = make_double2(0.0, 0.0); t3 = 0.0;
    if (l >= 2 && l <= d.lmax) {
        const double nl = __ldg(&d.spin2c[l].x);
        const double L = (double)l, M = (double)m;
        tp = make_double2(nl * (L - M * M), nl * (0.5 * L * (L - 1.0)));
        tm = make_double2(nl * (L - 1.0), 0.0);
        t3 = nl * sqrt((2.0 * L + 1.0) * (L - M) * (L + M) / (2.0 * L - 1.0));
    }
}

// ------------------------------------------------------------------------------------------------
// Staged-lambda mode (see sht_legendre.cu): F+/F- tiles written block by block to the plan's scratch, in the layout
// and order the contraction kernels consume them; same arithmetic as the fused generators (bit-identical tiles).
// ------------------------------------------------------------------------------------------------
static_assert(LAM_ABLK_BYTES == (size_t)A2_LBYTES && 2 * LAM_SBLK_BYTES == (size_t)S2_LBYTES, "block sizes");

// analysis block (m, l tile, chunk of 16 rings): [sign][class][ring][A2_SL]; warp = 32 l rows, lane = ring + 16 sign
__global__ void __launch_bounds__(128) k_fpm_blocks_analysis(DevicePlan d, double* __restrict__ lam)
{
    __shared__ __align__(16) double tile[A2_LBYTES / 8];
    __shared__ double2 cft[A2_ML], ctu[2 * A2_ML];
    __shared__ double ct3[A2_ML];
    const int m = blockIdx.y, lmax = d.lmax, nh = d.nh;
    const int t = blockIdx.x / d.nck_max, ck = blockIdx.x % d.nck_max;
    if (t > (lmax - m) / A2_ML) return;
    const int pc = d.pst[(size_t)m * d.ntile_max + t] + A2_PC * ck;
    if (pc >= nh) return;
    const size_t blk = (size_t)d.ablk_off[(size_t)m * d.ntile_max + t] + ck;
    const int lane = threadIdx.x & 31, gw = threadIdx.x >> 5;
    const int rr = lane & 15, sg = lane >> 4;
    const int l0 = m + t * A2_ML;
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    {
        const int l = l0 + threadIdx.x;
        double2 tp, tm; double t3;
        spin2_consts(d, l, m, tp, tm, t3);
        cft[threadIdx.x] = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        ctu[threadIdx.x] = tp; ctu[A2_ML + threadIdx.x] = tm; ct3[threadIdx.x] = t3;
    }
    for (int i = threadIdx.x; i < A2_LBYTES / 8; i += 128) tile[i] = 0.0;
    __syncthreads();
    constexpr int QL = A2_ML / 4;
    const int lq = l0 + QL * gw;
    const int p = pc + rr;
    double x1 = 0.0, x2 = 0.0, z = 0.0, is2 = 0.0;
    int ls = lmax + 1;
    if (p < nh && lq <= lmax) {
        const double2 sd = d.cseed[((size_t)d.csoff[m] + (lq - m) / LEG_CS) * nh + p];
        x1 = sd.x; x2 = sd.y; z = d.z[p]; is2 = 1.0 / d.sin2[p];
        ls = d.lstart[(size_t)m * nh + p];
    }
    const double ra = sg ? (double)m * z * is2 : is2;
    const double rc = sg ? (double)m * is2 : z * is2;
    const int rs = ls - lq;
    double* Ls = tile + (sg * 2 * A2_PC + rr) * A2_SL + (QL / 2) * gw;
    const double2* cfq = cft + QL * gw;
    const double2* tu = ctu + sg * A2_ML + QL * gw;
    const double* t3q = ct3 + QL * gw;
#pragma unroll 4
    for (int r = 0; r < QL; ++r) {
        const double2 ab = cfq[r];
        const double2 uv = tu[r];
        const double t3 = t3q[r];
        const double lamv = fma(ab.x * z, x1, -(ab.y * x2));
        const double U = fma(uv.x, ra, uv.y), W = t3 * rc;
        const double f = fma(lamv, U, -(x1 * W));
        const bool on = r >= rs;
        x2 = on ? x1 : x2; x1 = on ? lamv : x1;
        Ls[(r & 1) * (A2_PC * A2_SL) + (r >> 1)] = on ? f : 0.0;
    }
    __syncthreads();
    double2* dst = reinterpret_cast<double2*>(lam + blk * (size_t)(A2_LBYTES / 8));
    const double2* src = reinterpret_cast<const double2*>(tile);
    for (int i = threadIdx.x; i < A2_LBYTES / 16; i += 128) dst[i] = src[i];
}

// synthesis block (m, block of 64 rings, stage of 32 l): [sign][l][S2_SL]; 64 threads = rings, a thread forms F+ and F-
__global__ void __launch_bounds__(64) k_fpm_blocks_synthesis(DevicePlan d, double* __restrict__ lam)
{
    __shared__ double2 cab[S2_LC], ctp[S2_LC], ctm[S2_LC];
    const int m = blockIdx.z, pbi = blockIdx.y, n = blockIdx.x, lmax = d.lmax, nh = d.nh;
    const int cfirst = d.scfirst[(size_t)m * d.npb + pbi];
    const int lc = cfirst + S2_LC * n;
    if (cfirst > lmax || lc > lmax) return;
    const size_t blk = (size_t)d.sblk_off[(size_t)m * d.npb + pbi] + n;
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    if (threadIdx.x < S2_LC) {
        const int l = lc + threadIdx.x;
        double2 tp, tm; double t3;
        spin2_consts(d, l, m, tp, tm, t3);
        cab[threadIdx.x] = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        ctp[threadIdx.x] = tp; ctm[threadIdx.x] = make_double2(tm.x, t3);
    }
    __syncthreads();
    const int p = pbi * S2_PB + threadIdx.x;
    double x1 = 0.0, x2 = 0.0, z = 0.0, is2 = 0.0;
    int ls = lmax + 1;
    if (p < nh) {
        z = d.z[p]; is2 = 1.0 / d.sin2[p];
        ls = d.lstart[(size_t)m * nh + p];
        const double2 sd = d.cseed[((size_t)d.csoff[m] + (lc - m) / LEG_CS) * nh + p];
        x1 = sd.x; x2 = sd.y;
    }
    const double rap = is2, rcp = z * is2;
    const double ram = (double)m * z * is2, rcm = (double)m * is2;
    double* Lp = lam + blk * (size_t)(S2_LBYTES / 8) + threadIdx.x;
    double* Lm = Lp + S2_LC * S2_SL;
    const int rs = ls - lc;
#pragma unroll 4
    for (int r = 0; r < S2_LC; ++r) {
        const double2 ab = cab[r], tp = ctp[r], tm = ctm[r];
        const double lamv = fma(ab.x * z, x1, -(ab.y * x2));
        const double fp = fma(lamv, fma(tp.x, rap, tp.y), -(x1 * (tm.y * rcp)));
        const double fm = fma(lamv, tm.x * ram, -(x1 * (tm.y * rcm)));
        const bool on = r >= rs;
        x2 = on ? x1 : x2; x1 = on ? lamv : x1;
        Lp[r * S2_SL] = on ? fp : 0.0;
        Lm[r * S2_SL] = on ? fm : 0.0;
    }
    if (threadIdx.x < S2_SL - S2_PB)
        for (int r = 0; r < S2_LC; ++r) { Lp[r * S2_SL + S2_PB] = 0.0; Lm[r * S2_SL + S2_PB] = 0.0; }
}

// ------------------------------------------------------------------------------------------------
// analysis, spin 2: one CTA per (m, k-tile of 32 pairs); l tiles outer, ring chunks of 16 inner.
// Stage: [X: comp(Q,iU) x 8 kg x 16 p x 128 B, 128B-swizzled] [F: sign(+,-) x class x 16 p x A2_SL]
// ------------------------------------------------------------------------------------------------
// WHICH = 0: both a_E and a_B; 1: only a_E; 2: only a_B (item 9: half of the block products, output
// alm[map][nalm] of that component alone)
template <int WHICH>
__global__ void __launch_bounds__(LEG2_THREADS, 1)
k_legendre_analysis_spin2(const __grid_constant__ CUtensorMap tmF, DevicePlan d, double* __restrict__ alm, int k0, int kmaps,
                          int nkt, int accumulate, const double* __restrict__ lam, int m0, int tsplit, double* __restrict__ dout,
                          int pstar, int below)
{
    constexpr int nst = 3;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* stage_base = smem_raw;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)nst * A2_STAGE_BYTES);
    uint64_t* empty = full + 4;
    double2* cft = reinterpret_cast<double2*>(empty + 4);        // (alpha, beta) of the current l tile
    double2* ctu = cft + A2_ML;                                  // [sign][l]: (t1, t2) / (t4, 0)
    double* ct3 = reinterpret_cast<double*>(ctu + 2 * A2_ML);
    int* pst = reinterpret_cast<int*>(ct3 + A2_ML);

    // whole transform: one CTA per (m, k-tile), all l tiles.  Alg. 3 (tsplit = number of orders m0, m0 + 1, ..): one CTA
    // per (order, l tile, k-tile), as in the spin-0 kernel
    const int nt0 = (d.lmax - m0) / A2_ML + 1;
    const int m = tsplit ? m0 + blockIdx.x / (nkt * nt0) : m0 + blockIdx.x / nkt, kt = blockIdx.x % nkt;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lmax = d.lmax, nh = d.nh;
    const int ntile = (lmax - m) / A2_ML + 1;
    const int tb = tsplit ? (int)(blockIdx.x / nkt) % nt0 : 0, te = tsplit ? tb + 1 : ntile;
    if (tb >= ntile) return;
    // ring chunks of an l tile, split at the first chunk that starts at or past pstar (hybrid sweep of Alg. 3, as in the
    // spin-0 kernel): `below` = the chunks before it, else the chunks from it on; pstar = 0, below = 0: all chunks
    auto chunk_range = [&](int s, int& pb, int& pe) {
        const int cut = s >= pstar ? s : s + ((pstar - s + A2_PC - 1) / A2_PC) * A2_PC;
        pb = below ? s : cut;
        pe = below ? min(cut, nh) : nh;
    };

    for (int t = tid; t < ntile; t += LEG2_THREADS) pst[t] = d.pst[(size_t)m * d.ntile_max + t];
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) { mbar_init(full + s, lam ? 1 : 1 + 128); mbar_init(empty + s, LEG_CONSUMER_WARPS_S2); }
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();

    if (warp < 8) {
        // ===== consumers: (A^E, iA^B)[l, pair] += F+[l, p] (Q, iU)^{X(cls)}[p, pair] + F-[l, p] (iU, Q)^{X(1-cls)}[p, pair]
        const int cls = warp >> 2, wn = warp & 3;
        const int g = lane >> 2, t = lane & 3;
        double cE[8][2][2], cB[8][2][2];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) { cE[i][j][0] = cE[i][j][1] = 0.0; cB[i][j][0] = cB[i][j][1] = 0.0; }
        int stage = 0; uint32_t phase = 0;
        const size_t moff = (size_t)((long long)m * (2 * lmax + 1 - m) / 2);
        for (int tile = tb; tile < te; ++tile) {
            const int l0 = m + tile * A2_ML;
            const int i1 = min(8, (lmax - l0) / 16 + 1);        // 16-row blocks of the tile that reach down to l <= lmax
            int pcb, pce;
            chunk_range(pst[tile], pcb, pce);
            for (int pc = pcb; pc < pce; pc += A2_PC) {
                mbar_wait(full + stage, phase);
                const double* Xs = reinterpret_cast<const double*>(stage_base + (size_t)stage * A2_STAGE_BYTES);
                const double* Ls = Xs + A2_XBYTES / 8;
                // the first NI 16-row blocks: 8 except in the last tile, whose blocks past lmax are left out in steps of two
                auto contract = [&](auto ni_tag) {
                constexpr int NI = decltype(ni_tag)::value;
#pragma unroll
                for (int ks = 0; ks < A2_PC / 4; ++ks) {
                    const int pl = 8 * (ks >> 1) + 2 * t + (ks & 1);          // ring inside the 16-ring box
#pragma unroll
                    for (int sg = 0; sg < 2; ++sg) {
                        // sg = 0: F+ with the fold of this class; sg = 1: F- with the other fold and swapped components
                        const int h = cls ^ sg;
                        double a[NI], bq[2], bu[2];
                        const double* La = Ls + ((sg * 2 + cls) * A2_PC + pl) * A2_SL + g;
#pragma unroll
                        for (int i = 0; i < NI; ++i) a[i] = La[8 * i];
                        const double* Xb = Xs + pl * 16 + ((((4 * h + (g >> 1)) ^ (pl & 7)) << 1) | (g & 1));
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            bq[j] = Xb[(2 * wn + j) * 256];
                            bu[j] = Xb[(P_KG + 2 * wn + j) * 256];
                        }
#pragma unroll
                        for (int i = 0; i < NI; ++i)
#pragma unroll
                            for (int j = 0; j < 2; ++j) {
                                if (WHICH != 2) dmma884(cE[i][j][0], cE[i][j][1], a[i], sg ? bu[j] : bq[j]);
                                if (WHICH != 1) dmma884(cB[i][j][0], cB[i][j][1], a[i], sg ? bq[j] : bu[j]);
                            }
                    }
                }
                };
                if (i1 > 6) contract(std::integral_constant<int, 8>{});
                else if (i1 > 4) contract(std::integral_constant<int, 6>{});
                else if (i1 > 2) contract(std::integral_constant<int, 4>{});
                else contract(std::integral_constant<int, 2>{});
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + stage);
                if (++stage == nst) { stage = 0; phase ^= 1; }
            }
            // ---- epilogue: a_E = A^E, a_B = -i (iA^B), scattered to the m-major alm layout
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int l = l0 + 2 * (8 * i + g) + cls;
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int kk = kt * P_KT + (2 * wn + j) * KG + t;
                    if (l <= lmax && kk < kmaps) {
                        double2 ve = make_double2(cE[i][j][0], m == 0 ? 0.0 : cE[i][j][1]);
                        double2 vb = make_double2(cB[i][j][1], m == 0 ? 0.0 : -cB[i][j][0]);
                        if (WHICH == 0) {
                            double2* dst = reinterpret_cast<double2*>(alm) + ((size_t)(k0 + kk) * 2) * d.nalm + moff + l;
                            double2* dd = dout ? reinterpret_cast<double2*>(dout) + ((size_t)kk * 2) * d.nalm + moff + l : nullptr;
                            // all old values first: a load that follows a store through the same pointer is not moved above it
                            double2 de = make_double2(0.0, 0.0), db = de, ae = de, ab = de;
                            if (dd && below) { de = dd[0]; db = dd[d.nalm]; }     // the part from the ring pairs >= pstar
                            if (accumulate) { ae = dst[0]; ab = dst[d.nalm]; }
                            ve.x += de.x; ve.y += de.y; vb.x += db.x; vb.y += db.y;
                            if (dd) {                            // the increment itself, pairs indexed from the chunk start
                                dd[0] = ve;
                                dd[d.nalm] = vb;
                            }
                            ve.x += ae.x; ve.y += ae.y; vb.x += ab.x; vb.y += ab.y;
                            dst[0] = ve;
                            dst[d.nalm] = vb;
                        } else {
                            double2* dst = reinterpret_cast<double2*>(alm) + (size_t)(k0 + kk) * d.nalm + moff + l;
                            double2 v = WHICH == 1 ? ve : vb;
                            if (accumulate) { const double2 o = *dst; v.x += o.x; v.y += o.y; }
                            *dst = v;
                        }
                    }
                    cE[i][j][0] = cE[i][j][1] = 0.0; cB[i][j][0] = cB[i][j][1] = 0.0;
                }
            }
        }
    } else {
        // ===== generators (warps 8..11): every warp works on every chunk, warp g on the l rows [32 g, 32 g + 32) of the
        // tile (the recurrence restarts from the plan's state table every 16 l); lane = (ring 0..15) + 16 (sign of F).
        // Lane 0 of generator 0 also issues the TMA load of the chunk's Q / iU lines as soon as the stage is free.
        const int gw = warp - 8;
        if (lam) {
            // ===== staged mode: one thread streams, per stage, the chunk's Q / iU lines (TMA) and its F+/F- block (bulk copy)
            if (gw != 0 || lane != 0) return;
            int stage = 0; uint32_t phase = 0;
            for (int tile = tb; tile < te; ++tile) {
                const size_t blk0 = (size_t)d.ablk_off[(size_t)m * d.ntile_max + tile];
                int pcb, pce;
                chunk_range(pst[tile], pcb, pce);
                int ck = (pcb - pst[tile]) / A2_PC;
                for (int pc = pcb; pc < pce; pc += A2_PC, ++ck) {
                    mbar_wait(empty + stage, phase ^ 1);
                    unsigned char* Xs = stage_base + (size_t)stage * A2_STAGE_BYTES;
                    mbar_arrive_expect_tx(full + stage, A2_XBYTES + A2_LBYTES);
                    tma_load_4d(Xs, &tmF, full + stage, 0, pc, kt * P_KG, m * 2);
                    bulk_load(Xs + A2_XBYTES, lam + (blk0 + ck) * (size_t)(A2_LBYTES / 8), A2_LBYTES, full + stage);
                    if (++stage == nst) { stage = 0; phase ^= 1; }
                }
            }
            return;
        }
        const int rr = lane & 15, sg = lane >> 4;
        const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
        const double2* csm = d.cseed + (size_t)d.csoff[m] * nh;
        constexpr int QL = A2_ML / 4;                           // l rows per generator warp
        // per-l constants of the next tile: one l per generator thread, fetched while the current tile is computed
        const int gl = gw * 32 + lane;
        double2 nab, ntp, ntm; double nt3;
        auto load_consts = [&](int l0) {
            const int l = l0 + gl;
            nab = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
            spin2_consts(d, l, m, ntp, ntm, nt3);
        };
        load_consts(m + tb * A2_ML);
        int stage = 0; uint32_t phase = 0;
        for (int tile = tb; tile < te; ++tile) {
            const int l0 = m + tile * A2_ML;
            named_bar_sync(1, 128);                             // every generator is done with the previous tile
            cft[gl] = nab; ctu[gl] = ntp; ctu[A2_ML + gl] = ntm; ct3[gl] = nt3;
            named_bar_sync(1, 128);
            if (tile + 1 < te) load_consts(l0 + A2_ML);
            const int lq = l0 + QL * gw;                        // first l of this warp's quarter
            const double2* cst = csm + (size_t)((lq - m) / LEG_CS) * nh;
            int pcb, pce;
            chunk_range(pst[tile], pcb, pce);
            for (int pc = pcb; pc < pce; pc += A2_PC) {
                const int p = pc + rr;
                double x1 = 0.0, x2 = 0.0, z = 0.0, is2 = 0.0;
                int ls = lmax + 1;
                if (p < nh && lq <= lmax) {
                    const double2 sd = __ldg(cst + p);
                    x1 = sd.x; x2 = sd.y; z = d.z[p]; is2 = 1.0 / d.sin2[p];
                    ls = d.lstart[(size_t)m * nh + p];
                }
                const double ra = sg ? (double)m * z * is2 : is2;       // multiplies t1 (F+) / t4 (F-)
                const double rc = sg ? (double)m * is2 : z * is2;       // multiplies t3
                const int rs = ls - lq;
                mbar_wait(empty + stage, phase ^ 1);
                unsigned char* Xs = stage_base + (size_t)stage * A2_STAGE_BYTES;
                if (gw == 0 && lane == 0) {
                    mbar_arrive_expect_tx(full + stage, A2_XBYTES);
                    tma_load_4d(Xs, &tmF, full + stage, 0, pc, kt * P_KG, m * 2);
                }
                double* Ls = reinterpret_cast<double*>(Xs + A2_XBYTES) + (sg * 2 * A2_PC + rr) * A2_SL + (QL / 2) * gw;
                const double2* cfq = cft + QL * gw;
                const double2* tu = ctu + sg * A2_ML + QL * gw;
                const double* t3q = ct3 + QL * gw;
#pragma unroll 8
                for (int r = 0; r < QL; ++r) {
                    const double2 ab = cfq[r];
                    const double2 uv = tu[r];
                    const double t3 = t3q[r];
                    const double lam = fma(ab.x * z, x1, -(ab.y * x2));
                    const double U = fma(uv.x, ra, uv.y), W = t3 * rc;
                    const double f = fma(lam, U, -(x1 * W));             // x1 = lambda_{l-1}
                    const bool on = r >= rs;
                    x2 = on ? x1 : x2; x1 = on ? lam : x1;
                    Ls[(r & 1) * (A2_PC * A2_SL) + (r >> 1)] = on ? f : 0.0;
                }
                mbar_arrive(full + stage);
                if (++stage == nst) { stage = 0; phase ^= 1; }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// synthesis, spin 2: one CTA per (m, block of 64 ring pairs, k-tile of 32 pairs); loops over l chunks of 32.
// Stage: [a_lm: 4 boxes (8 l each) x comp(E,B) x 32 pairs x 128 B, 128B-swizzled] [F: sign x 32 l x S2_SL]
// With Qe = sum_{l-m even} F+ A^E + sum_{l-m odd} F- iA^B (even under the fold) and Qo the complementary sums,
// Q(north) = Qe + Qo, Q(south) = Qe - Qo; iU likewise with A^E and iA^B exchanged.
// ------------------------------------------------------------------------------------------------
// WHICH = 0: alm holds (a_E, a_B) per pair; 1 / 2: alm[map][nalm] holds only a_E / only a_B, the other one is zero
template <int WHICH, bool ORD = false>
__global__ void __launch_bounds__(LEG2_THREADS, 1)
k_legendre_synthesis_spin2(const __grid_constant__ CUtensorMap tmA, DevicePlan d, double* __restrict__ F, int k0, int kmaps,
                           int nkt, int npb, const double* __restrict__ lam, int m0, int nsplit, int pb0, int pb1)
{
    constexpr int NST = 3;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* stage_base = smem_raw;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + NST * S2_STAGE_BYTES);
    uint64_t* empty = full + 4;
    double2* cfs = reinterpret_cast<double2*>(empty + 4);       // 4 generator warps x 2 buffers x S2_LC x (ab, uv, t3)

    // the CTA walks its share of the ring blocks of (m, k-tile) back to back, the pipeline running across them (see the
    // spin-0 kernel): whole transforms nsplit = 1, the one-order launches of Alg. 3 one block per CTA
    const int kt = blockIdx.x % nkt;
    const int sp = (blockIdx.x / nkt) % nsplit;
    // ORD: a few orders at a time from m0 (Alg. 3); a separate instantiation keeps the whole-transform kernel's registers
    const int m = (ORD ? m0 : 0) + blockIdx.x / (nkt * nsplit);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lmax = d.lmax, nh = d.nh;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(full + s, lam ? 1 : 1 + 128); mbar_init(empty + s, LEG_CONSUMER_WARPS_S2); }
        fence_barrier_init();
        tma_prefetch_desc(&tmA);
    }
    __syncthreads();
    const size_t moff = (size_t)((long long)m * (2 * lmax + 1 - m) / 2);
    const int* scf = d.scfirst + (size_t)m * npb;

    if (warp < 8) {
        // ===== consumers: warp (par, wn): rows = 64 rings of the even (par 0) / odd (par 1) fold part, 8 pairs =====
        const int par = warp >> 2, wn = warp & 3;
        const int g = lane >> 2, t = lane & 3;
        double cQ[8][2][2], cU[8][2][2];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) { cQ[i][j][0] = cQ[i][j][1] = 0.0; cU[i][j][0] = cU[i][j][1] = 0.0; }
        int stage = 0; uint32_t phase = 0;
        const int im = g & 1;
        const bool zero_e = (m == 0) && im;               // Im(a_l0) is ignored
        const bool zero_b = (m == 0) && !im;
        // per-lane offsets (doubles): F rows of the 4 l of a step with sign sg, a_lm element of pair j for sign sg
        const int la0 = (2 * t + par) * S2_SL + g;                             // sg = 0: class = par
        const int la1 = (S2_LC + 2 * t + (par ^ 1)) * S2_SL + g;               // sg = 1: class = 1 - par
        const int c0 = par, c1 = par ^ 1;
        int ab0[2], ab1[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int pr = 8 * wn + 4 * j + (g >> 1);                          // pair inside the k-tile
            ab0[j] = pr * 16 + (((2 * t + par) ^ (pr & 7)) << 1);
            ab1[j] = pr * 16 + (((2 * t + (par ^ 1)) ^ (pr & 7)) << 1);
        }
        // this lane's workspace cell of (ring g, pairs 4 (8 kt + 2 wn) + t .., Q, fold part par); + i: 8 rings, + j: 4 pairs
        const size_t kgs = (size_t)(lmax + 1) * 2 * 2 * KG, ps = (size_t)d.nkg * kgs;
        double2* Fl = reinterpret_cast<double2*>(F) + f_cell(d, g, kt * P_KG + wn * 2, m, 0, par) + t;
        for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
        const int pb = pbi * S2_PB;
        if (m >= d.mlim[min(pb + S2_PB, nh) - 1]) continue;       // no ring of this block takes part in order m (never read)
        for (int lc = scf[pbi]; lc <= lmax; lc += S2_LC) {
            mbar_wait(full + stage, phase);
            const double* As = reinterpret_cast<const double*>(stage_base + (size_t)stage * S2_STAGE_BYTES);
            const double* Ls = As + S2_ABYTES / 8;
            const int lrow = lc + 2 * t - 2;                // (l - 2) of this lane's first row of box 0, without the class bit
            const int ks1 = min(S2_LC / 4, 2 * ((lmax - lc) / 8 + 1));          // boxes of 8 l that reach down to l <= lmax
#pragma unroll
            for (int ks = 0; ks < S2_LC / 4; ++ks) {
                if (ks >= ks1) break;
                // box q of 8 l; sg = 0: the 4 l whose class matches this warp's fold part (F+), sg = 1: the others (F-)
                const int q = ks >> 1, sg = ks & 1;
                double a[8], be[2], bb[2];
                const double* La = Ls + (sg ? la1 : la0) + 8 * q * S2_SL;
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = La[8 * i];
                // rows outside 2 <= l <= lmax are not this order's input: l < 2 is ignored (reading G13) and the tail of
                // the last chunk holds the next order's first entries (its ignored l < 2 slots among them)
                const bool dead = (unsigned)(lrow + 8 * q + (sg ? c1 : c0)) > (unsigned)(lmax - 2);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const double* Ab = As + q * 1024 + (sg ? ab1[j] : ab0[j]);
                    const double e = Ab[im];                    // A^E: (re, im) of a_E
                    const double b = Ab[(WHICH == 2 ? 0 : P_KT * 16) + (im ^ 1)];  // iA^B = (-Im a_B, Re a_B)
                    be[j] = (dead || zero_e) ? 0.0 : e;
                    bb[j] = (dead || zero_b) ? 0.0 : (im ? b : -b);
                }
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        if (WHICH == 0) {
                            dmma884(cQ[i][j][0], cQ[i][j][1], a[i], sg ? bb[j] : be[j]);
                            dmma884(cU[i][j][0], cU[i][j][1], a[i], sg ? be[j] : bb[j]);
                        } else if (WHICH == 1) {                // a_B = 0: Q takes F+ A^E, iU takes F- A^E
                            if (sg) dmma884(cU[i][j][0], cU[i][j][1], a[i], be[j]);
                            else dmma884(cQ[i][j][0], cQ[i][j][1], a[i], be[j]);
                        } else {                                // a_E = 0: Q takes F- iA^B, iU takes F+ iA^B
                            if (sg) dmma884(cQ[i][j][0], cQ[i][j][1], a[i], bb[j]);
                            else dmma884(cU[i][j][0], cU[i][j][1], a[i], bb[j]);
                        }
                    }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + stage);
            if (++stage == NST) { stage = 0; phase ^= 1; }
        }
        // ---- epilogue: the even (par 0) / odd (par 1) fold parts go straight from the accumulators into the two halves of
        // the workspace lines of Q and iU; north = e + o, south = e - o are formed by the ring kernels on load
        double2* Fb = Fl + (size_t)pb * ps;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const bool inr = pb + 8 * i + g < nh;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (inr) {
                    double2* dst = Fb + (size_t)(8 * i) * ps + (size_t)j * kgs;
                    dst[0] = make_double2(cQ[i][j][0], cQ[i][j][1]);
                    dst[2 * KG] = make_double2(cU[i][j][0], cU[i][j][1]);
                }
                cQ[i][j][0] = cQ[i][j][1] = 0.0; cU[i][j][0] = cU[i][j][1] = 0.0;
            }
        }
        }
    } else {
        // ===== generators (warps 8..11): warp = (half of the 64 rings) + 2 (half of the stage's 32 l); a lane forms F+
        // and F- of its ring; the recurrence restarts from the plan's state table every 16 l.  Lane 0 of generator 0
        // issues the TMA loads of a_E / a_B for the stage.
        const int gw = warp - 8;
        if (lam) {
            // ===== staged mode: one thread streams, per stage, the a_E / a_B boxes (TMA) and the F+/F- block (bulk copy)
            if (gw != 0 || lane != 0) return;
            int stage = 0; uint32_t phase = 0;
            for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
                if (m >= d.mlim[min(pbi * S2_PB + S2_PB, nh) - 1]) continue;
                const size_t blk0 = (size_t)d.sblk_off[(size_t)m * d.npb + pbi];
                int n = 0;
                for (int lc = scf[pbi]; lc <= lmax; lc += S2_LC, ++n) {
                    mbar_wait(empty + stage, phase ^ 1);
                    unsigned char* As = stage_base + (size_t)stage * S2_STAGE_BYTES;
                    mbar_arrive_expect_tx(full + stage, S2_ABYTES + S2_LBYTES);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        tma_load_3d(As + q * (S2_ABYTES / 4), &tmA, full + stage, (int)(2 * (moff + lc + 8 * q)), k0 + kt * P_KT, 0);
                    bulk_load(As + S2_ABYTES, lam + (blk0 + n) * (size_t)(S2_LBYTES / 8), S2_LBYTES, full + stage);
                    if (++stage == NST) { stage = 0; phase ^= 1; }
                }
            }
            return;
        }
        const int gh = gw >> 1;
        const int rl = (gw & 1) * 32 + lane;
        int stage = 0, buf = 0; uint32_t phase = 0;
        const int row0 = k0 + kt * P_KT;
        for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
        const int pb = pbi * S2_PB;
        if (m >= d.mlim[min(pb + S2_PB, nh) - 1]) continue;
        const int cfirst = scf[pbi];
        const int p = pb + rl;
        double z = 0.0, is2 = 0.0;
        int ls = lmax + 1;
        if (p < nh) { ls = d.lstart[(size_t)m * nh + p]; z = d.z[p]; is2 = 1.0 / d.sin2[p]; }
        const double rap = is2, rcp = z * is2;                               // F+: multiply t1, t3
        const double ram = (double)m * z * is2, rcm = (double)m * is2;       // F-: multiply t4, t3
        const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
        const double2* csm = d.cseed + (size_t)d.csoff[m] * nh + (p < nh ? p : 0);
        constexpr int HL = S2_LC / 2;                           // l per warp and stage
        double2* cfw = cfs + gw * (2 * HL * 3);
        double2 nab, ntp, ntm; double nt3;
        auto load_consts = [&](int lb) {
            const int l = lb + (lane & (HL - 1));
            nab = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
            spin2_consts(d, l, m, ntp, ntm, nt3);
        };
        auto load_state = [&](int lb) -> double2 {
            return (p < nh && lb <= lmax) ? __ldg(csm + (size_t)((lb - m) / LEG_CS) * nh) : make_double2(0.0, 0.0);
        };
        load_consts(cfirst + HL * gh);
        double2 sd = load_state(cfirst + HL * gh);
        for (int lc = cfirst; lc <= lmax; lc += S2_LC) {
            const int lb = lc + HL * gh;
            double2* cb = cfw + buf * (HL * 3);
            if (lane < HL) { cb[lane] = nab; cb[HL + lane] = make_double2(ntp.x, ntp.y); cb[2 * HL + lane] = make_double2(ntm.x, nt3); }
            __syncwarp();
            double x1 = sd.x, x2 = sd.y;
            load_consts(lb + S2_LC);
            sd = load_state(lb + S2_LC);
            const int rs = ls - lb;
            mbar_wait(empty + stage, phase ^ 1);
            unsigned char* As = stage_base + (size_t)stage * S2_STAGE_BYTES;
            if (gw == 0 && lane == 0) {
                mbar_arrive_expect_tx(full + stage, S2_ABYTES);
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    tma_load_3d(As + q * (S2_ABYTES / 4), &tmA, full + stage, (int)(2 * (moff + lc + 8 * q)), row0, 0);
            }
            double* Lp = reinterpret_cast<double*>(As + S2_ABYTES) + (HL * gh) * S2_SL + rl;
            double* Lm = Lp + S2_LC * S2_SL;
#pragma unroll
            for (int r = 0; r < HL; ++r) {
                const double2 ab = cb[r];
                const double2 tp = cb[HL + r];                  // (t1, t2)
                const double2 tm = cb[2 * HL + r];              // (t4, t3)
                const double lam = fma(ab.x * z, x1, -(ab.y * x2));
                const double fp = fma(lam, fma(tp.x, rap, tp.y), -(x1 * (tm.y * rcp)));      // x1 = lambda_{l-1}
                const double fm = fma(lam, tm.x * ram, -(x1 * (tm.y * rcm)));
                const bool on = r >= rs;
                x2 = on ? x1 : x2; x1 = on ? lam : x1;
                Lp[r * S2_SL] = on ? fp : 0.0;
                Lm[r * S2_SL] = on ? fm : 0.0;
            }
            mbar_arrive(full + stage);
            buf ^= 1;
            if (++stage == NST) { stage = 0; phase ^= 1; }
        }
        }
    }
}

// ---- host side -------------------------------------------------------------------------------------------
// alm[pair][comp][nalm*2 doubles] as a 3-D tensor (innermost first: doubles of one (pair, comp) row, pair, comp);
// box = 8 l (128 bytes) x 32 pairs x (E, B): lands in shared memory as [comp][pair][128 B]
static cudaError_t make_tmap_alm_spin2(const DevicePlan& d, const double* alm, long long pairs, int ncomp_mem, CUtensorMap* tm)
{
    // ncomp_mem = 1: single-component a_lm (E-only / B-only transforms): the box's second component is out of bounds
    // and arrives as zeros
    const cuuint64_t dims[3] = {(cuuint64_t)d.nalm * 2, (cuuint64_t)pairs, (cuuint64_t)ncomp_mem};
    const cuuint64_t strides[2] = {(cuuint64_t)d.nalm * 16 * ncomp_mem, (cuuint64_t)d.nalm * 16};
    const cuuint32_t box[3] = {16, P_KT, 2};
    return make_tmap_f64(tm, alm, 3, dims, strides, box);
}

static size_t analysis2_smem(int ntile)
{
    return (size_t)3 * A2_STAGE_BYTES + 8 * sizeof(uint64_t) + (size_t)A2_ML * (3 * sizeof(double2) + sizeof(double)) +
           (size_t)ntile * sizeof(int);
}
static size_t synthesis2_smem()
{
    return (size_t)3 * S2_STAGE_BYTES + 8 * sizeof(uint64_t) + (size_t)4 * 2 * S2_LC * 3 * sizeof(double2) + 16;
}

cudaError_t launch_lambda_blocks_spin2(sht_plan_s* pl, const DevicePlan& d, bool analysis, cudaStream_t st)
{
    if (!(pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam)) return cudaSuccess;
    if (analysis) {
        k_fpm_blocks_analysis<<<dim3((unsigned)(d.ntile_max * d.nck_max), (unsigned)(d.lmax + 1)), 128, 0, st>>>(d, pl->lam);
        pl->launches++;
    } else if (d.nst_max > 0) {
        k_fpm_blocks_synthesis<<<dim3((unsigned)d.nst_max, (unsigned)d.npb, (unsigned)(d.lmax + 1)), 64, 0, st>>>(d, pl->lam);
        pl->launches++;
    }
    return cudaGetLastError();
}

cudaError_t launch_legendre_analysis_spin2(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                           bool accumulate, cudaStream_t st, int pol, bool gen_lambda, int pstar)
{
    const size_t sm = analysis2_smem(d.ntile_max);
    auto kern = pol == 1 ? k_legendre_analysis_spin2<1> : pol == 2 ? k_legendre_analysis_spin2<2> : k_legendre_analysis_spin2<0>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tmF;
    if ((e = make_tmap_F(d, F, P_KG, 2, &tmF)) != cudaSuccess) return e;
    const int nkt = (kmaps + P_KT - 1) / P_KT;
    const bool staged = pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam;
    if (staged && gen_lambda && (e = launch_lambda_blocks_spin2(pl, d, true, st)) != cudaSuccess) return e;
    kern<<<(d.lmax + 1) * nkt, LEG2_THREADS, sm, st>>>(tmF, d, alm, k0, kmaps, nkt, accumulate ? 1 : 0, staged ? pl->lam : nullptr, 0, 0, nullptr,
                                                       pstar, 0);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_legendre_synthesis_spin2(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps,
                                            cudaStream_t st, int pol, bool gen_lambda, int pb0)
{
    const size_t sm = synthesis2_smem();
    auto kern = pol == 1 ? k_legendre_synthesis_spin2<1> : pol == 2 ? k_legendre_synthesis_spin2<2> : k_legendre_synthesis_spin2<0>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tmA;
    if ((e = make_tmap_alm_spin2(d, alm, (long long)(k0 + kmaps), pol ? 1 : 2, &tmA)) != cudaSuccess) return e;
    const int nkt = (kmaps + P_KT - 1) / P_KT;
    const int npb = (d.nh + S2_PB - 1) / S2_PB;
    const bool staged = pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam;
    if (staged && gen_lambda && (e = launch_lambda_blocks_spin2(pl, d, false, st)) != cudaSuccess) return e;
    kern<<<(d.lmax + 1) * nkt, LEG2_THREADS, sm, st>>>(tmA, d, F, k0, kmaps, nkt, npb, staged ? pl->lam : nullptr, 0, 1, pb0, npb);
    pl->launches++;
    return cudaGetLastError();
}

// ---- a few orders at a time (Alg. 3): the spin-2 side of the per-order launchers of sht_legendre.cu
cudaError_t legendre_order_maps_spin2(const DevicePlan& d, const double* F, const double* da, int kmaps, CUtensorMap* tmF, CUtensorMap* tmA)
{
    cudaError_t e = cudaFuncSetAttribute(k_legendre_analysis_spin2<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)analysis2_smem(d.ntile_max));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_legendre_synthesis_spin2<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)synthesis2_smem());
    if (e == cudaSuccess) e = make_tmap_F(d, F, P_KG, 2, tmF);
    if (e == cudaSuccess) e = make_tmap_alm_spin2(d, da, (long long)kmaps, 2, tmA);
    return e;
}

cudaError_t launch_legendre_analysis_order_spin2(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmF, double* alm, double* da,
                                                 int k0, int kmaps, int m, int nm, cudaStream_t st, int pstar)
{
    const int nkt = (kmaps + P_KT - 1) / P_KT;
    const int ntile = (d.lmax - m) / A2_ML + 1;
    k_legendre_analysis_spin2<0><<<(unsigned)(nm * ntile * nkt), LEG2_THREADS, analysis2_smem(d.ntile_max), st>>>(tmF, d, alm, k0, kmaps, nkt, 1,
                                                                                                                 nullptr, m, nm, da, pstar, pstar > 0 ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_legendre_synthesis_order_spin2(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmA, double* F, int kmaps, int m,
                                                  int nm, cudaStream_t st, int pbend)
{
    const int nkt = (kmaps + P_KT - 1) / P_KT;
    const int npb = (d.nh + S2_PB - 1) / S2_PB;
    const int nb = pbend > 0 && pbend < npb ? pbend : npb;
    k_legendre_synthesis_spin2<0, true><<<(unsigned)(nm * nkt * nb), LEG2_THREADS, synthesis2_smem(), st>>>(tmA, d, F, 0, kmaps, nkt, npb, nullptr, m, nb,
                                                                                                           0, nb);
    pl->launches++;
    return cudaGetLastError();
}

}  // namespace sht
