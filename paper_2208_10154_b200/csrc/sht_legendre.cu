// sht_legendre.cu -- subsystem (2): fused Legendre recurrence + FP64 tensor-core (DMMA.8x8x4) contraction,
// and subsystem (3): the m-major a_lm scatter / gather in its epilogue / prologue.
//
//   analysis  (PAPER.md:56-60 eq. 3, :95 eq. 7):  A_m = P_m T_m, contraction over ring pairs p,
//       a_lm^k = sum_p lambda_lm(theta_p) X_p^k,  X = E (l+m even) or O (l+m odd)   [N/S fold]
//   synthesis (PAPER.md:74-76 eq. 5, :97 eq. 7):  T_m = P_m^t A_m, contraction over l,
//       Ee_p = sum_{l+m even} lambda_lm(theta_p) a_lm,  Oo_p likewise; north = Ee + Oo, south = Ee - Oo.
//
// Both kernels are warp specialised (12 warps): 8 consumer warps issue DMMA on a 128 x 128 CTA tile (each warp
// 64 x 32, accumulators in registers -- FP64 has no tcgen05/TMEM path on sm_100a, DMMA.8x8x4 is the native FP64
// tensor instruction), one producer warp streams the operand tiles (T_m^k(theta) resp. a_lm) with TMA
// (cp.async.bulk.tensor, 128-byte swizzle) into an mbarrier-guarded ring of shared-memory stages, and generator
// warps run the three-term recurrence from the plan's l_safe(m,p) (item 11)
// into the same stages.  The lambda tile and the operand tile of a stage are released together by the consumers.
// Rings whose lambda is below threshold for a whole tile are skipped (ring optimisation, item 10, :229).
#include <type_traits>
#include <cstdio>
#include "sht_legendre_common.cuh"

namespace sht {

// ---- tile shapes ---------------------------------------------------------------------------------------
constexpr int LEG_GEN_WARPS = 4;             // lambda generators (+ TMA issue)
constexpr int LEG_CONSUMER_WARPS = 8;        // 2 (l parity class) x 4 (32-column slices); warp tile 64 x 32
constexpr int LEG_THREADS = 384;             // + warp 8: TMA producer, warps 9,10: lambda generators, warp 11 idle
constexpr int A_ML = LEG_A_ML;               // analysis: l rows per tile (64 of each parity class)
constexpr int A_PC = 32;                     // analysis: ring pairs per stage (two TMA boxes of 16)
constexpr int A_SL = 66;                     // lambda tile: stride (doubles) between rings, = 2 mod 8: conflict-free A fragments
constexpr int A_STAGES = 2;
constexpr int A_XBYTES = A_PC * NK * 2 * 8;  // E and O rows of a stage: 64 KB
constexpr int A_LBYTES = 2 * A_PC * A_SL * 8;
constexpr int A_STAGE_BYTES = A_XBYTES + A_LBYTES;
static_assert(A_STAGE_BYTES % 1024 == 0, "stages must keep the 1024-byte alignment of the swizzled TMA boxes");
constexpr int S_PB = 64;                     // synthesis: ring pairs per CTA tile (Ee rows + Oo rows = 128 C rows)
constexpr int S_LC = 32;                     // synthesis: l values per stage (16 of each parity, four TMA boxes of 8 l)
constexpr int S_SL = 66;                     // lambda tile: stride (doubles) between l rows, = 2 mod 8
constexpr int S_STAGES = 4;                  // even: the generators fill stages in pairs
constexpr int S_ABYTES = S_LC * KTILE_MAPS * 16;     // a_lm tile of a stage: 32 KB
constexpr int S_LBYTES = S_LC * S_SL * 8;
constexpr int S_STAGE_BYTES = (S_ABYTES + S_LBYTES + 1023) / 1024 * 1024;

// ------------------------------------------------------------------------------------------------
// Staged-lambda mode: the lambda tiles of one transform, written block by block to an HBM scratch in exactly the
// layout and order the contraction kernels consume them (same recurrence, same seeds, same arithmetic as the fused
// generators: bit-identical tiles).  Here the scalar FP64 work runs at the full DFMA rate, away from the DMMA pipe.
// ------------------------------------------------------------------------------------------------
static_assert(LAM_ABLK_BYTES == (size_t)A_LBYTES && LAM_SBLK_BYTES == (size_t)S_LBYTES, "block sizes");

// Rows of a lambda tile below the smallest l_safe of a group of 8 rings hold zeros for those rings: the consumers skip their
// 16-row blocks.  One nibble per group of 8 lanes (= rings of the chunk): the first 16-row block (0..8) with a started
// recurrence; called by a full warp with its lanes' l_safe.
__device__ __forceinline__ int pack_i0(int ls, int l0)
{
    int lsmin = ls;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) lsmin = min(lsmin, __shfl_xor_sync(0xffffffffu, lsmin, o));
    const int v = max(0, min(8, (lsmin - l0) >> 4));
    return __shfl_sync(0xffffffffu, v, 0) | (__shfl_sync(0xffffffffu, v, 8) << 4) | (__shfl_sync(0xffffffffu, v, 16) << 8) |
           (__shfl_sync(0xffffffffu, v, 24) << 12);
}

// analysis block (m, l tile, chunk of 32 rings): [class][ring][A_SL]; 128 threads: warp = 32 l rows, lane = ring
__global__ void __launch_bounds__(128) k_lambda_blocks_analysis(DevicePlan d, double* __restrict__ lam, int* __restrict__ i0tab)
{
    __shared__ __align__(16) double tile[2 * A_PC * A_SL];
    const int m = blockIdx.y, lmax = d.lmax, nh = d.nh;
    const int t = blockIdx.x / d.nck_max, ck = blockIdx.x % d.nck_max;
    if (t > (lmax - m) / A_ML) return;
    const int pc = d.pst[(size_t)m * d.ntile_max + t] + A_PC * ck;
    if (pc >= nh) return;
    const size_t blk = (size_t)d.ablk_off[(size_t)m * d.ntile_max + t] + ck;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int l0 = m + t * A_ML, lw = l0 + 32 * w;
    const int p = pc + lane;
    for (int i = threadIdx.x; i < 2 * A_PC * A_SL; i += 128) tile[i] = 0.0;      // padding columns included
    __syncthreads();
    double x1 = 0.0, x2 = 0.0, z = 0.0;
    int ls = lmax + 1;
    if (p < nh) {
        z = d.z[p];
        ls = d.lstart[(size_t)m * nh + p];
        if (lw <= lmax) {
            const double2 sd = d.cseed[((size_t)d.csoff[m] + (lw - m) / LEG_CS) * nh + p];
            x1 = sd.x; x2 = sd.y;
        }
    }
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    const int rs = ls - lw;
#pragma unroll 4
    for (int r = 0; r < 32; ++r) {
        const int l = lw + r;
        const double2 ab = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        const double tv = fma(ab.x * z, x1, -(ab.y * x2));
        const bool on = r >= rs;
        x2 = on ? x1 : x2; x1 = on ? tv : x1;
        const int rr = 32 * w + r;
        tile[(rr & 1) * (A_PC * A_SL) + lane * A_SL + (rr >> 1)] = on ? tv : 0.0;
    }
    if (w == 0) {                                           // per 8 rings: first 16-row block with a started recurrence
        const int pk = pack_i0(ls, l0);
        if (lane == 0) i0tab[blk] = pk;
    }
    __syncthreads();
    double2* dst = reinterpret_cast<double2*>(lam + blk * (size_t)(A_LBYTES / 8));
    const double2* src = reinterpret_cast<const double2*>(tile);
    for (int i = threadIdx.x; i < A_LBYTES / 16; i += 128) dst[i] = src[i];
}

// synthesis block (m, block of 64 rings, stage of 32 l): [l][S_SL]; 64 threads = rings (stores are coalesced over rings)
__global__ void __launch_bounds__(64) k_lambda_blocks_synthesis(DevicePlan d, double* __restrict__ lam)
{
    const int m = blockIdx.z, pbi = blockIdx.y, n = blockIdx.x, lmax = d.lmax, nh = d.nh;
    const int cfirst = d.scfirst[(size_t)m * d.npb + pbi];
    const int lc = cfirst + S_LC * n;
    if (cfirst > lmax || lc > lmax) return;
    const size_t blk = (size_t)d.sblk_off[(size_t)m * d.npb + pbi] + n;
    const int p = pbi * S_PB + threadIdx.x;
    double x1 = 0.0, x2 = 0.0, z = 0.0;
    int ls = lmax + 1;
    if (p < nh) {
        z = d.z[p];
        ls = d.lstart[(size_t)m * nh + p];
        const double2 sd = d.cseed[((size_t)d.csoff[m] + (lc - m) / LEG_CS) * nh + p];
        x1 = sd.x; x2 = sd.y;
    }
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    double* dst = lam + blk * (size_t)(S_LBYTES / 8) + threadIdx.x;
    const int rs = ls - lc;
#pragma unroll 4
    for (int r = 0; r < S_LC; ++r) {
        const int l = lc + r;
        const double2 ab = l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        const double tv = fma(ab.x * z, x1, -(ab.y * x2));
        const bool on = r >= rs;
        x2 = on ? x1 : x2; x1 = on ? tv : x1;
        dst[r * S_SL] = on ? tv : 0.0;
    }
    if (threadIdx.x < S_SL - S_PB)                          // padding columns
        for (int r = 0; r < S_LC; ++r) dst[r * S_SL + S_PB] = 0.0;
}

// ------------------------------------------------------------------------------------------------
// analysis kernel: one CTA per (m, k-tile); l tiles outer, ring chunks inner.
// Stage layout: [X: 2 boxes x (16 kg x 16 p x 128 B, 128B-swizzled)] [lambda: 2 classes x 32 p x A_SL]
// ------------------------------------------------------------------------------------------------
// WIN = 1 (per-order launches of Alg. 3): four CTAs share an l tile, each owns a window of two 16-row blocks (32 l) -- the
// launch has a few dozen CTAs for 148 SMs, so the tile is cut up for parallelism; its own instantiation, so that the
// whole-transform kernel (WIN = 0) keeps its code and register allocation
template <int WIN>
__global__ void __launch_bounds__(LEG_THREADS, 1)
k_legendre_analysis(const __grid_constant__ CUtensorMap tmF, DevicePlan d, double* __restrict__ alm, int k0, int kmaps,
                    int nkt, int accumulate, const double* __restrict__ lam, const int* __restrict__ i0tab,
                    int m0, int tsplit, double* __restrict__ dout, int pstar, int below)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* stage_base = smem_raw;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + A_STAGES * A_STAGE_BYTES);
    uint64_t* empty = full + A_STAGES;
    double2* cft = reinterpret_cast<double2*>(empty + A_STAGES);                           // (alpha, beta) of the current l tile
    int* pst = reinterpret_cast<int*>(cft + A_ML);                                         // first ring of every l tile
    int* i0s = pst + ((d.ntile_max + 3) & ~3);                                               // per stage: first 16-row block with a started recurrence

    // whole transform: one CTA per (m, k-tile), all l tiles.  A few orders at a time (Alg. 3, tsplit = number of orders
    // m0, m0 + 1, ..): one CTA per (order, l tile, k-tile) -- the tiles restart from the state table, so they are
    // independent; the grid is sized for the tiles of m0, the CTAs past the last tile of their order leave
    // tsplit > 0: tile-split mode, tsplit = l tiles per CTA (the grid is sized for the tile groups of order m0)
    const int nt0 = ((d.lmax - m0) / A_ML + tsplit) / (tsplit > 0 ? tsplit : 1);
    const int wsel = WIN ? (int)(blockIdx.x & 3) : 0, ib = 2 * wsel;       // WIN: this CTA's window = row blocks ib, ib + 1
    const unsigned bx = WIN ? blockIdx.x >> 2 : blockIdx.x;
    const int m = tsplit ? m0 + bx / (nkt * nt0) : m0 + bx / nkt, kt = bx % nkt;
    // warps 0..3 generate (the oldest warps of an SM sub-partition are served first by its scheduler: their
    // FP64 instructions must slip in between the consumers' DMMAs), warps 4..11 consume
    const int lane = threadIdx.x & 31, warp = (threadIdx.x >> 5) - LEG_GEN_WARPS;
    const int tix = threadIdx.x;
    const int lmax = d.lmax, nh = d.nh;
    const int comp = 0;
    const int ntile = (lmax - m) / A_ML + 1;
    const int tb = tsplit ? ((int)(bx / nkt) % nt0) * tsplit : 0, te = tsplit ? min(tb + tsplit, ntile) : ntile;
    if (tb >= ntile) return;
    if (WIN && ib >= min(8, (d.lmax - (m + tb * A_ML)) / 16 + 1)) return;      // the window lies past lmax
    // ring chunks of an l tile: A_PC ring pairs from the tile's first ring pst on.  Alg. 3 (hybrid sweep) splits them at the
    // first chunk that starts at or past pstar: `below` = the chunks before it (they hold every ring pair < pstar), else
    // the chunks from it on (ring pairs >= pstar only).  pstar = 0, below = 0: all chunks.
    auto chunk_range = [&](int s, int& pb, int& pe) {
        const int cut = s >= pstar ? s : s + ((pstar - s + A_PC - 1) / A_PC) * A_PC;
        pb = below ? s : cut;
        pe = below ? min(cut, nh) : nh;
    };

    for (int t = tix; t < ntile; t += LEG_THREADS) pst[t] = d.pst[(size_t)m * d.ntile_max + t];
    if (tix == 0) {
        for (int s = 0; s < A_STAGES; ++s) { mbar_init(full + s, lam ? 1 : 1 + 64); mbar_init(empty + s, LEG_CONSUMER_WARPS); }
        fence_barrier_init();
        tma_prefetch_desc(&tmF);
    }
    __syncthreads();

    if (warp >= 0) {
        // ===== consumers: C[l, k'] += lambda[l, p] X[p, k'] =====
        const int cls = warp >> 2, wn = warp & 3;      // cls 0: l - m even (uses E), 1: odd (uses O)
        const int g = lane >> 2, t = lane & 3;
        double c[8][4][2];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) { c[i][j][0] = 0.0; c[i][j][1] = 0.0; }
        int stage = 0; uint32_t phase = 0;
        const size_t moff = (size_t)((long long)m * (2 * lmax + 1 - m) / 2);
        for (int tile = tb; tile < te; ++tile) {
            const int l0 = m + tile * A_ML;
            const int i1 = min(8, (lmax - l0) / 16 + 1);        // 16-row blocks of the tile that reach down to l <= lmax
            int pcb, pce;
            chunk_range(pst[tile], pcb, pce);
            for (int pc = pcb; pc < pce; pc += A_PC) {
                mbar_wait(full + stage, phase);
                const double* Xs = reinterpret_cast<const double*>(stage_base + (size_t)stage * A_STAGE_BYTES);
                const double* Ls = Xs + A_XBYTES / 8 + cls * (A_PC * A_SL);
                // rows below the smallest l_safe of 8 rings hold lambda = 0 for them: their 16-row blocks (i < i0) are skipped
                const int i0p = i0s[stage];
                if constexpr (WIN != 0) {
#pragma unroll
                    for (int ks = 0; ks < A_PC / 4; ++ks) {
                        const int sub = ks >> 2, ksl = ks & 3;
                        const int pl = 8 * (ksl >> 1) + 2 * t + (ksl & 1);
                        const int i0 = (i0p >> (4 * (2 * sub + (ksl >> 1)))) & 15;
                        double a[2], b[4];
                        const double* La = Ls + (16 * sub + pl) * A_SL + g;
                        const double* Xb = Xs + sub * 4096 + pl * 16 + ((((4 * cls + (g >> 1)) ^ (pl & 7)) << 1) | (g & 1));
#pragma unroll
                        for (int i = 0; i < 2; ++i) a[i] = La[8 * (ib + i)];
#pragma unroll
                        for (int j = 0; j < 4; ++j) b[j] = Xb[(4 * wn + j) * 256];
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            if (ib + i >= i0 && ib + i < i1) {
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
                            }
                        }
                    }
                } else
                if (i0p == 0) {
                    // plain loop over the first NI 16-row blocks (NI = 8 except in the last tile, whose blocks past lmax
                    // are left out in steps of two: a block-by-block test costs more than the blocks it saves)
                    auto contract = [&](auto ni_tag) {
                        constexpr int NI = decltype(ni_tag)::value;
#pragma unroll
                        for (int ks = 0; ks < A_PC / 4; ++ks) {
                            const int sub = ks >> 2, ksl = ks & 3;
                            const int pl = 8 * (ksl >> 1) + 2 * t + (ksl & 1);        // ring inside the 16-ring box
                            double a[NI], b[4];
                            const double* La = Ls + (16 * sub + pl) * A_SL + g;
#pragma unroll
                            for (int i = 0; i < NI; ++i) a[i] = La[8 * i];
                            const double* Xb = Xs + sub * 4096 + pl * 16 + ((((4 * cls + (g >> 1)) ^ (pl & 7)) << 1) | (g & 1));
#pragma unroll
                            for (int j = 0; j < 4; ++j) b[j] = Xb[(4 * wn + j) * 256];
#pragma unroll
                            for (int i = 0; i < NI; ++i)
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
                        }
                    };
                    if (i1 > 6) contract(std::integral_constant<int, 8>{});
                    else if (i1 > 4) contract(std::integral_constant<int, 6>{});
                    else if (i1 > 2) contract(std::integral_constant<int, 4>{});
                    else contract(std::integral_constant<int, 2>{});
                } else {
#pragma unroll
                    for (int ks = 0; ks < A_PC / 4; ++ks) {
                        const int sub = ks >> 2, ksl = ks & 3;
                        const int pl = 8 * (ksl >> 1) + 2 * t + (ksl & 1);
                        const int i0 = (i0p >> (4 * (2 * sub + (ksl >> 1)))) & 15;       // the 8 rings this step draws from
                        double b[4];
                        const double* La = Ls + (16 * sub + pl) * A_SL + g;
                        const double* Xb = Xs + sub * 4096 + pl * 16 + ((((4 * cls + (g >> 1)) ^ (pl & 7)) << 1) | (g & 1));
#pragma unroll
                        for (int j = 0; j < 4; ++j) b[j] = Xb[(4 * wn + j) * 256];
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            if (i >= i0 && i < i1) {
                                const double a = La[8 * i];
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a, b[j]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + stage);
                if (++stage == A_STAGES) { stage = 0; phase ^= 1; }
            }
            // ---- epilogue: scatter to the m-major alm layout; a lane holds (re, im) of one (l, map)
            // (the old values of two maps of a row are loaded together before anything is stored: a load that follows
            // a store through the same pointer cannot be moved above it, and 32 dependent round trips to HBM per tile were
            // a fifth of the accumulating launches of Alg. 2 and most of the per-order launches of Alg. 3)
            const bool rd_d = dout != nullptr && below, rd_a = accumulate != 0;
            if constexpr (WIN != 0) {
                // the window's 32 l x 64 maps through the (drained) stage buffers, then one cooperative read-modify-write:
                // eight elements per thread, consecutive threads on consecutive l of one map
                double2* T = reinterpret_cast<double2*>(stage_base);
                constexpr int WR = 32, TROW = WR + 1;
                named_bar_sync(2, LEG_CONSUMER_WARPS * 32);
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        T[(wn * 16 + 4 * j + t) * TROW + 16 * i + 2 * g + cls] = make_double2(c[i][j][0], m == 0 ? 0.0 : c[i][j][1]);
                named_bar_sync(2, LEG_CONSUMER_WARPS * 32);
                const int ct = tix - LEG_GEN_WARPS * 32;
                const int lw = l0 + 16 * ib;                         // first l of the window
                const int nl = min(WR, lmax - lw + 1), nk = min(KTILE_MAPS, kmaps - kt * KTILE_MAPS);
                constexpr int EB = KTILE_MAPS * WR / (LEG_CONSUMER_WARPS * 32);      // 8
                double2 od[EB], oa[EB];
#pragma unroll
                for (int u = 0; u < EB; ++u) {
                    const int e = ct + u * LEG_CONSUMER_WARPS * 32, kl = e / WR, ll = e % WR;
                    od[u] = make_double2(0.0, 0.0); oa[u] = make_double2(0.0, 0.0);
                    if (kl < nk && ll < nl) {
                        const int kk = kt * KTILE_MAPS + kl;
                        if (rd_d) od[u] = reinterpret_cast<const double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + lw + ll];
                        if (rd_a) oa[u] = reinterpret_cast<const double2*>(alm)[((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + lw + ll];
                    }
                }
#pragma unroll
                for (int u = 0; u < EB; ++u) {
                    const int e = ct + u * LEG_CONSUMER_WARPS * 32, kl = e / WR, ll = e % WR;
                    if (kl < nk && ll < nl) {
                        const int kk = kt * KTILE_MAPS + kl;
                        double2 v = T[kl * TROW + ll];
                        v.x += od[u].x; v.y += od[u].y;
                        if (dout) reinterpret_cast<double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + lw + ll] = v;
                        v.x += oa[u].x; v.y += oa[u].y;
                        reinterpret_cast<double2*>(alm)[((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + lw + ll] = v;
                    }
                }
                continue;                                            // one tile per CTA in this mode
            }
            if ((rd_d || rd_a) && tile == te - 1) {
                // Last tile of the CTA (the only one of a per-order launch): the pipeline has drained, so the stage buffers
                // are free.  The tile goes through shared memory ([map][l], rows padded by one element) and the consumer
                // warps do the read-modify-write together: consecutive threads take consecutive l of one map (coalesced),
                // and every thread has its eight loads in flight before its first store.
                double2* T = reinterpret_cast<double2*>(stage_base);
                constexpr int TROW = A_ML + 1;
                named_bar_sync(2, LEG_CONSUMER_WARPS * 32);          // every consumer warp is done reading the last stage
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        T[(wn * 16 + 4 * j + t) * TROW + 2 * (8 * i + g) + cls] = make_double2(c[i][j][0], m == 0 ? 0.0 : c[i][j][1]);
                        c[i][j][0] = 0.0; c[i][j][1] = 0.0;
                    }
                named_bar_sync(2, LEG_CONSUMER_WARPS * 32);
                const int ct = tix - LEG_GEN_WARPS * 32;             // 0 .. 255
                const int nl = min(A_ML, lmax - l0 + 1), nk = min(KTILE_MAPS, kmaps - kt * KTILE_MAPS);
                constexpr int EB = 8;                                // elements per thread and batch
                for (int e0 = ct; e0 < KTILE_MAPS * A_ML; e0 += EB * LEG_CONSUMER_WARPS * 32) {
                    double2 od[EB], oa[EB];
#pragma unroll
                    for (int u = 0; u < EB; ++u) {
                        const int e = e0 + u * LEG_CONSUMER_WARPS * 32, kl = e / A_ML, ll = e % A_ML;
                        od[u] = make_double2(0.0, 0.0); oa[u] = make_double2(0.0, 0.0);
                        if (kl < nk && ll < nl) {
                            const int kk = kt * KTILE_MAPS + kl;
                            if (rd_d) od[u] = reinterpret_cast<const double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + l0 + ll];
                            if (rd_a) oa[u] = reinterpret_cast<const double2*>(alm)[((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + l0 + ll];
                        }
                    }
#pragma unroll
                    for (int u = 0; u < EB; ++u) {
                        const int e = e0 + u * LEG_CONSUMER_WARPS * 32, kl = e / A_ML, ll = e % A_ML;
                        if (kl < nk && ll < nl) {
                            const int kk = kt * KTILE_MAPS + kl;
                            double2 v = T[kl * TROW + ll];
                            v.x += od[u].x; v.y += od[u].y;
                            if (dout) reinterpret_cast<double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + l0 + ll] = v;
                            v.x += oa[u].x; v.y += oa[u].y;
                            reinterpret_cast<double2*>(alm)[((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + l0 + ll] = v;
                        }
                    }
                }
                continue;                                            // (the loop over the tiles ends here)
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int l = l0 + 2 * (8 * i + g) + cls;
#pragma unroll
                for (int jh = 0; jh < 4; jh += 2) {               // two maps at a time: the register budget has no room for four
                    double2 od[2], oa[2];
#pragma unroll
                    for (int jj = 0; jj < 2; ++jj) {
                        const int kk = kt * KTILE_MAPS + wn * 16 + 4 * (jh + jj) + t;
                        od[jj] = make_double2(0.0, 0.0); oa[jj] = make_double2(0.0, 0.0);
                        if (l <= lmax && kk < kmaps) {
                            if (rd_d) od[jj] = reinterpret_cast<const double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + l];
                            if (rd_a) oa[jj] = reinterpret_cast<const double2*>(alm)[((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + l];
                        }
                    }
#pragma unroll
                    for (int jj = 0; jj < 2; ++jj) {
                        const int j = jh + jj;
                        const int kk = kt * KTILE_MAPS + wn * 16 + 4 * j + t;
                        if (l <= lmax && kk < kmaps) {
                            double2* dst = reinterpret_cast<double2*>(alm) + ((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + moff + l;
                            // the increment (+ the part from the ring pairs >= pstar, hybrid sweep), then the accumulated a_lm
                            double2 v = make_double2(c[i][j][0] + od[jj].x, (m == 0 ? 0.0 : c[i][j][1]) + od[jj].y);
                            if (dout)                            // rows indexed from the chunk start
                                reinterpret_cast<double2*>(dout)[((size_t)kk * d.ncomp + comp) * d.nalm + moff + l] = v;
                            v.x += oa[jj].x; v.y += oa[jj].y;
                            *dst = v;
                        }
                        c[i][j][0] = 0.0; c[i][j][1] = 0.0;
                    }
                }
            }
        }
    } else {
        // ===== lambda generators (warps 8..11): warp = (stage it owns) + 2 (half of the tile's 128 l rows); lane = ring of
        // the chunk.  The recurrence restarts from the plan's state table at l0 and l0 + 64, so the two halves of a
        // stage are generated at the same time.  Lane 0 of the first-half warp also issues the stage's TMA loads.
        const int gw = warp + LEG_GEN_WARPS;
        if (lam) {
            // ===== staged mode: one thread streams, per stage, the chunk's operand lines (TMA) and its lambda block (bulk
            // copy from the scratch the generator kernel filled), and hands the consumers the block's first active row
            if (gw != 0 || lane != 0) return;
            int chunk = 0;
            for (int tile = tb; tile < te; ++tile) {
                const size_t blk0 = (size_t)d.ablk_off[(size_t)m * d.ntile_max + tile];
                int pcb, pce;
                chunk_range(pst[tile], pcb, pce);
                int ck = (pcb - pst[tile]) / A_PC;
                for (int pc = pcb; pc < pce; pc += A_PC, ++chunk, ++ck) {
                    const int stage = chunk & 1;
                    const uint32_t phase = (chunk >> 1) & 1;
                    const int i0v = __ldg(i0tab + blk0 + ck);
                    mbar_wait(empty + stage, phase ^ 1);
                    unsigned char* Xs = stage_base + (size_t)stage * A_STAGE_BYTES;
                    i0s[stage] = i0v;
                    mbar_arrive_expect_tx(full + stage, A_XBYTES + A_LBYTES);
                    tma_load_4d(Xs, &tmF, full + stage, 0, pc, kt * (KTILE_MAPS / KG), m * d.ncomp + comp);
                    tma_load_4d(Xs + A_XBYTES / 2, &tmF, full + stage, 0, pc + 16, kt * (KTILE_MAPS / KG), m * d.ncomp + comp);
                    bulk_load(Xs + A_XBYTES, lam + (blk0 + ck) * (size_t)(A_LBYTES / 8), A_LBYTES, full + stage);
                }
            }
            return;
        }
        const int gs = gw & 1, gh = gw >> 1;
        const int gl = gw * 32 + lane;                          // 0 .. 127 = one l of the tile per thread
        const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
        const double2* csm = d.cseed + (size_t)d.csoff[m] * nh;
        // (alpha, beta) of an l tile are staged in shared memory once per tile (a dependent global load per
        // recurrence step would cost an L2 round trip per l); rows past lmax get (0, 0)
        auto load_cf = [&](int l0) -> double2 {
            const int l = l0 + gl;
            return l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        };
        double2 cf0 = load_cf(m + tb * A_ML);
        int chunk = 0;
        for (int tile = tb; tile < te; ++tile) {
            const int l0 = m + tile * A_ML;
            named_bar_sync(1, 128);                             // every generator is done with the previous tile
            cft[gl] = cf0;
            named_bar_sync(1, 128);
            if (tile + 1 < te) cf0 = load_cf(l0 + A_ML);
            const int lh = l0 + (A_ML / 2) * gh;                // first l of this warp's half
            const double2* cst = csm + (size_t)((lh - m) / LEG_CS) * nh;
            int pcb, pce;
            chunk_range(pst[tile], pcb, pce);
            for (int pc = pcb; pc < pce; pc += A_PC, ++chunk) {
                if ((chunk & 1) != gs) continue;
                const int stage = gs;
                const uint32_t phase = (chunk >> 1) & 1;
                // NCH independent chains per lane (16 l each, restarted from the state table): a dependent FP64 instruction
                // waits behind the consumers' queued DMMAs for hundreds of cycles, so the latency of one step is shared
                // by four chains instead of being paid 64 times in a row
                constexpr int NCH = 4, CL = A_ML / 2 / NCH;
                const int p = pc + lane;
                double x1[NCH], x2[NCH], z = 0.0;
                int ls = lmax + 1;
#pragma unroll
                for (int c = 0; c < NCH; ++c) { x1[c] = 0.0; x2[c] = 0.0; }
                if (p < nh) {
                    z = d.z[p];
                    ls = d.lstart[(size_t)m * nh + p];
#pragma unroll
                    for (int c = 0; c < NCH; ++c) {
                        if (lh + CL * c <= lmax) {
                            const double2 sd = __ldg(cst + (size_t)c * (CL / LEG_CS) * nh + p);
                            x1[c] = sd.x; x2[c] = sd.y;
                        }
                    }
                }
                const int rs = ls - lh;                             // first row of the half with a started recurrence
                const int i0pk = pack_i0(ls, l0);
                mbar_wait(empty + stage, phase ^ 1);
                unsigned char* Xs = stage_base + (size_t)stage * A_STAGE_BYTES;
                if (gh == 0 && lane == 0) {
                    i0s[stage] = i0pk;
                    mbar_arrive_expect_tx(full + stage, A_XBYTES);
                    tma_load_4d(Xs, &tmF, full + stage, 0, pc, kt * (KTILE_MAPS / KG), m * d.ncomp + comp);
                    tma_load_4d(Xs + A_XBYTES / 2, &tmF, full + stage, 0, pc + 16, kt * (KTILE_MAPS / KG), m * d.ncomp + comp);
                }
                double* Ls = reinterpret_cast<double*>(Xs + A_XBYTES) + lane * A_SL + (A_ML / 4) * gh;
                const double2* cfh = cft + (A_ML / 2) * gh;
#pragma unroll
                for (int r = 0; r < CL; ++r) {
#pragma unroll
                    for (int c = 0; c < NCH; ++c) {
                        const int rr = CL * c + r;                  // row inside this warp's half
                        const double2 ab = cfh[rr];
                        const double t = fma(ab.x * z, x1[c], -(ab.y * x2[c]));
                        const bool on = rr >= rs;
                        const double v = on ? t : 0.0;
                        x2[c] = on ? x1[c] : x2[c]; x1[c] = on ? t : x1[c];
                        Ls[(rr & 1) * (A_PC * A_SL) + (rr >> 1)] = v;
                    }
                }
                mbar_arrive(full + stage);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// synthesis kernel: one CTA per (m, k-tile, share of the blocks of 64 ring pairs); per block it loops over l chunks of
// 32.  The CTA walks its ring blocks back to back: the mbarrier pipeline keeps running across them (the generators
// fill the stages of the next block while the consumers finish and store the current one), so its fill and drain are
// paid once per CTA instead of once per block.  Whole transforms give a CTA all blocks of (m, k-tile) (nsplit = 1);
// the one-order launches of Alg. 3 spread the blocks over nsplit CTAs.
// The even sum Ee (l - m even) and the odd sum Oo of a ring pair are stored as they leave the accumulators, in the two
// halves of the pair's workspace line; north = Ee + Oo and south = Ee - Oo are formed by the ring kernels on load.
// Stage layout: [a_lm: 4 boxes x (64 maps x 8 l x 16 B, 128B-swizzled)] [lambda: 32 l x S_SL]
// ------------------------------------------------------------------------------------------------
// WIN = 1 (per-order launches of Alg. 3): four CTAs share a block of 64 ring pairs, each owns two of its eight 8-ring row
// blocks, as in k_legendre_analysis<1>
template <int WIN>
__global__ void __launch_bounds__(LEG_THREADS, 1)
k_legendre_synthesis(const __grid_constant__ CUtensorMap tmA, DevicePlan d, double* __restrict__ F, int k0, int kmaps,
                     int nkt, int npb, const double* __restrict__ lam, int m0, int nsplit, int pb0, int pb1)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* stage_base = smem_raw;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + S_STAGES * S_STAGE_BYTES);
    uint64_t* empty = full + S_STAGES;
    double2* cfs = reinterpret_cast<double2*>(empty + S_STAGES);      // 4 generator warps x 2 buffers x S_LC/2 (alpha, beta)

    // block order: m slowest (long m first), then the share of ring blocks, k-tile fastest
    const int ib = WIN ? 2 * (int)(blockIdx.x & 3) : 0;             // WIN: this CTA's row blocks ib, ib + 1 of every ring block
    const unsigned bx = WIN ? blockIdx.x >> 2 : blockIdx.x;
    const int kt = bx % nkt;
    const int sp = (bx / nkt) % nsplit;
    const int m = m0 + bx / (nkt * nsplit);
    // warps 0..3 generate (the oldest warps of an SM sub-partition are served first by its scheduler: their
    // FP64 instructions must slip in between the consumers' DMMAs), warps 4..11 consume
    const int lane = threadIdx.x & 31, warp = (threadIdx.x >> 5) - LEG_GEN_WARPS;
    const int tix = threadIdx.x;
    const int lmax = d.lmax, nh = d.nh;
    const int comp = 0;

    if (tix == 0) {
        for (int s = 0; s < S_STAGES; ++s) { mbar_init(full + s, lam ? 1 : 1 + 128); mbar_init(empty + s, LEG_CONSUMER_WARPS); }
        fence_barrier_init();
        tma_prefetch_desc(&tmA);
    }
    __syncthreads();
    const size_t moff = (size_t)((long long)m * (2 * lmax + 1 - m) / 2);
    const int* scf = d.scfirst + (size_t)m * npb;

    if (warp >= 0) {
        // ===== consumers: C[p, k'] += lambda[l, p] a[l, k'] over the l of this warp's parity class =====
        const int cls = warp >> 2, wn = warp & 3;
        const int g = lane >> 2, t = lane & 3;
        double c[8][4][2];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) { c[i][j][0] = 0.0; c[i][j][1] = 0.0; }
        int stage = 0; uint32_t phase = 0;
        const bool kill_im = (m == 0) && (g & 1);      // Im(a_l0) is ignored
        // this lane's workspace cell of (ring pb + g, maps 4 (16 kt + 4 wn) + t .., half cls); + i: 8 rings, + j: 4 maps
        const size_t kgs = (size_t)(lmax + 1) * d.ncomp * 2 * KG, ps = (size_t)d.nkg * kgs;
        double2* Fl = reinterpret_cast<double2*>(F) + f_cell(d, g, kt * (KTILE_MAPS / KG) + wn * 4, m, comp, cls) + t;
        for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
            const int pb = pbi * S_PB;
            if (m >= d.mlim[min(pb + S_PB, nh) - 1]) continue;        // no ring of this block takes part in order m (never read)
            const int cfirst = scf[pbi];
            // smallest l_safe of every 8-ring row block
            const int4 q0 = __ldg(reinterpret_cast<const int4*>(d.sminls8 + ((size_t)m * npb + pbi) * 8));
            const int4 q1 = __ldg(reinterpret_cast<const int4*>(d.sminls8 + ((size_t)m * npb + pbi) * 8 + 4));
            for (int lc = cfirst; lc <= lmax; lc += S_LC) {
                mbar_wait(full + stage, phase);
                const double* As = reinterpret_cast<const double*>(stage_base + (size_t)stage * S_STAGE_BYTES);
                const double* Ls = As + S_ABYTES / 8;
                // 8-ring row blocks whose recurrences all start after this stage hold lambda = 0: skipped
                auto active = [&](int lend) -> unsigned {
                    return (q0.x <= lend ? 1u : 0u) | (q0.y <= lend ? 2u : 0u) | (q0.z <= lend ? 4u : 0u) | (q0.w <= lend ? 8u : 0u) |
                           (q1.x <= lend ? 16u : 0u) | (q1.y <= lend ? 32u : 0u) | (q1.z <= lend ? 64u : 0u) | (q1.w <= lend ? 128u : 0u);
                };
                const int ks1 = min(S_LC / 8, (lmax - lc) / 8 + 1);          // steps of 8 l that reach down to l <= lmax
                if constexpr (WIN != 0) {
#pragma unroll
                    for (int ks = 0; ks < S_LC / 8; ++ks) {
                        if (ks >= ks1) break;
                        const unsigned act = active(lc + 8 * ks + 7);
                        double a[2], b[4];
                        const double* La = Ls + (8 * ks + 2 * t + cls) * S_SL + g;
#pragma unroll
                        for (int i = 0; i < 2; ++i) a[i] = La[8 * (ib + i)];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int row = 16 * wn + 4 * j + (g >> 1);
                            const double v = As[ks * 1024 + row * 16 + ((((2 * t + cls) ^ (row & 7)) << 1) | (g & 1))];
                            b[j] = kill_im ? 0.0 : v;
                        }
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            if (act & (1u << (ib + i))) {
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
                            }
                        }
                    }
                } else
                if (active(lc + 7) == 0xffu && ks1 == S_LC / 8) {  // every recurrence has started by the first 8 l of the stage
#pragma unroll
                    for (int ks = 0; ks < S_LC / 8; ++ks) {
                        double a[8], b[4];
                        const double* La = Ls + (8 * ks + 2 * t + cls) * S_SL + g;
#pragma unroll
                        for (int i = 0; i < 8; ++i) a[i] = La[8 * i];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int row = 16 * wn + 4 * j + (g >> 1);               // map inside the k-tile
                            const double v = As[ks * 1024 + row * 16 + ((((2 * t + cls) ^ (row & 7)) << 1) | (g & 1))];
                            b[j] = kill_im ? 0.0 : v;
                        }
#pragma unroll
                        for (int i = 0; i < 8; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
                    }
                } else {
#pragma unroll
                    for (int ks = 0; ks < S_LC / 8; ++ks) {
                        if (ks >= ks1) break;
                        const unsigned act = active(lc + 8 * ks + 7);               // the step's 8 l: lc + 8 ks ..
                        double b[4];
                        const double* La = Ls + (8 * ks + 2 * t + cls) * S_SL + g;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int row = 16 * wn + 4 * j + (g >> 1);
                            const double v = As[ks * 1024 + row * 16 + ((((2 * t + cls) ^ (row & 7)) << 1) | (g & 1))];
                            b[j] = kill_im ? 0.0 : v;
                        }
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            if (act & (1u << i)) {
                                const double a = La[8 * i];
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a, b[j]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + stage);
                if (++stage == S_STAGES) { stage = 0; phase ^= 1; }
            }
            // ---- epilogue: a lane holds (re, im) of (ring pb + 8 i + g, map 16 wn + 4 j + t): 64-byte runs per ring
            double2* Fb = Fl + (size_t)pb * ps;
#pragma unroll
            for (int i = 0; i < (WIN ? 2 : 8); ++i) {
                const int ig = ib + i;                                       // row block inside the ring block
                const bool inr = pb + 8 * ig + g < nh;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (inr) Fb[(size_t)(8 * ig) * ps + (size_t)j * kgs] = make_double2(c[i][j][0], c[i][j][1]);
                    c[i][j][0] = 0.0; c[i][j][1] = 0.0;
                }
            }
        }
    } else {
        // ===== lambda generators (warps 0..3): warp = (half of the block's 64 rings) + 2 (half of the stage's 32 l);
        // the recurrence restarts from the plan's state table every 16 l, so the two l halves of a stage are generated
        // at the same time.  Lane 0 of generator 0 also issues the stage's TMA loads (a_lm, straight from the m-major
        // ABI layout).
        const int gw = warp + LEG_GEN_WARPS;
        if (lam) {
            // ===== staged mode: one thread streams, per stage, the a_lm boxes (TMA) and the lambda block (bulk copy)
            if (gw != 0 || lane != 0) return;
            const int row0s = (k0 + kt * KTILE_MAPS) * d.ncomp + comp;
            int stage = 0; uint32_t phase = 0;
            for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
                if (m >= d.mlim[min(pbi * S_PB + S_PB, nh) - 1]) continue;
                const size_t blk0 = (size_t)d.sblk_off[(size_t)m * d.npb + pbi];
                int n = 0;
                for (int lc = scf[pbi]; lc <= lmax; lc += S_LC, ++n) {
                    mbar_wait(empty + stage, phase ^ 1);
                    unsigned char* As = stage_base + (size_t)stage * S_STAGE_BYTES;
                    mbar_arrive_expect_tx(full + stage, S_ABYTES + S_LBYTES);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        tma_load_2d(As + q * (S_ABYTES / 4), &tmA, full + stage, (int)(2 * (moff + lc + 8 * q)), row0s);
                    bulk_load(As + S_ABYTES, lam + (blk0 + n) * (size_t)(S_LBYTES / 8), S_LBYTES, full + stage);
                    if (++stage == S_STAGES) { stage = 0; phase ^= 1; }
                }
            }
            return;
        }
        const int gh = gw >> 1;
        const int rl = (gw & 1) * 32 + lane;
        const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
        constexpr int HL = S_LC / 2;                            // l per warp and stage
        double2* cfw = cfs + gw * (2 * HL);                     // this warp's coefficients of the two stages
        auto load_cf = [&](int lb) -> double2 {                 // lanes 0..15: first stage of the pair, 16..31: second
            const int l = lb + (lane & (HL - 1)) + (lane >> 4) * S_LC;
            return l <= lmax ? __ldg(coefm + l) : make_double2(0.0, 0.0);
        };
        int stage = 0; uint32_t phase = 0;
        const int row0 = (k0 + kt * KTILE_MAPS) * d.ncomp + comp;
        for (int pbi = pb0 + sp; pbi < pb1; pbi += nsplit) {
            const int pb = pbi * S_PB;
            if (m >= d.mlim[min(pb + S_PB, nh) - 1]) continue;
            const int cfirst = scf[pbi];
            const int p = pb + rl;
            double z = 0.0;
            int ls = lmax + 1;
            if (p < nh) { ls = d.lstart[(size_t)m * nh + p]; z = d.z[p]; }
            const double2* csm = d.cseed + (size_t)d.csoff[m] * nh + (p < nh ? p : 0);
            auto load_state = [&](int lb) -> double2 {
                return (p < nh && lb <= lmax) ? __ldg(csm + (size_t)((lb - m) / LEG_CS) * nh) : make_double2(0.0, 0.0);
            };
            // Two stages are generated at a time, as two independent chains per lane (restarted from the state table): a
            // dependent FP64 instruction waits behind the consumers' queued DMMAs for hundreds of cycles, so the latency
            // of a step is shared by both chains.  (alpha, beta) and the start states of the next pair are fetched while
            // the current pair is computed.
            const int lb0 = cfirst + HL * gh;
            double2 cf = load_cf(lb0), sda = load_state(lb0), sdb = load_state(lb0 + S_LC);
            for (int lc = cfirst; lc <= lmax; lc += 2 * S_LC) {
                const int lb = lc + HL * gh;
                const bool two = lc + S_LC <= lmax;             // the pair's second stage exists
                __syncwarp();                                   // everyone is done reading the previous coefficients
                cfw[lane] = cf;
                __syncwarp();
                double xa1 = sda.x, xa2 = sda.y, xb1 = sdb.x, xb2 = sdb.y;
                cf = load_cf(lb + 2 * S_LC); sda = load_state(lb + 2 * S_LC); sdb = load_state(lb + 3 * S_LC);
                const int rsa = ls - lb, rsb = rsa - S_LC;
                // a block with an odd number of stages leaves the pairs of the next block on an odd stage: the second
                // stage of a pair may be the wrapped one
                const int stb = stage + 1 == S_STAGES ? 0 : stage + 1;
                const uint32_t phb = stb == 0 ? phase ^ 1 : phase;
                mbar_wait(empty + stage, phase ^ 1);
                if (two) mbar_wait(empty + stb, phb ^ 1);
                unsigned char* Asa = stage_base + (size_t)stage * S_STAGE_BYTES;
                unsigned char* Asb = stage_base + (size_t)stb * S_STAGE_BYTES;
                if (gw == 0 && lane == 0) {
                    mbar_arrive_expect_tx(full + stage, S_ABYTES);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        tma_load_2d(Asa + q * (S_ABYTES / 4), &tmA, full + stage, (int)(2 * (moff + lc + 8 * q)), row0);
                    if (two) {
                        mbar_arrive_expect_tx(full + stb, S_ABYTES);
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            tma_load_2d(Asb + q * (S_ABYTES / 4), &tmA, full + stb, (int)(2 * (moff + lc + S_LC + 8 * q)), row0);
                    }
                }
                double* La = reinterpret_cast<double*>(Asa + S_ABYTES) + (HL * gh) * S_SL + rl;
                double* Lb = reinterpret_cast<double*>(Asb + S_ABYTES) + (HL * gh) * S_SL + rl;
                if (two) {
#pragma unroll
                    for (int r = 0; r < HL; ++r) {
                        const double2 aa = cfw[r], ab = cfw[HL + r];
                        const double ta = fma(aa.x * z, xa1, -(aa.y * xa2));
                        const double tb = fma(ab.x * z, xb1, -(ab.y * xb2));
                        const bool ona = r >= rsa, onb = r >= rsb;
                        xa2 = ona ? xa1 : xa2; xa1 = ona ? ta : xa1;
                        xb2 = onb ? xb1 : xb2; xb1 = onb ? tb : xb1;
                        La[r * S_SL] = ona ? ta : 0.0;
                        Lb[r * S_SL] = onb ? tb : 0.0;
                    }
                    mbar_arrive(full + stage);
                    mbar_arrive(full + stb);
                } else {
#pragma unroll
                    for (int r = 0; r < HL; ++r) {
                        const double2 aa = cfw[r];
                        const double ta = fma(aa.x * z, xa1, -(aa.y * xa2));
                        const bool ona = r >= rsa;
                        xa2 = ona ? xa1 : xa2; xa1 = ona ? ta : xa1;
                        La[r * S_SL] = ona ? ta : 0.0;
                    }
                    mbar_arrive(full + stage);
                }
                stage += two ? 2 : 1;
                if (stage >= S_STAGES) { stage -= S_STAGES; phase ^= 1; }
            }
        }
    }
}

// ---- host side: tensor maps and launches ---------------------------------------------------------------
// alm[row = map*ncomp+comp][nalm*2 doubles] as a 2-D tensor; box = 8 l (128 bytes) x 64 rows
static cudaError_t make_tmap_alm(const DevicePlan& d, const double* alm, long long rows, CUtensorMap* tm)
{
    const cuuint64_t dims[2] = {(cuuint64_t)d.nalm * 2, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)d.nalm * 16};
    const cuuint32_t box[2] = {16, KTILE_MAPS};
    return make_tmap_f64(tm, alm, 2, dims, strides, box);
}

static size_t analysis_smem(int ntile)
{
    return (size_t)A_STAGES * A_STAGE_BYTES + 2 * A_STAGES * sizeof(uint64_t) + (size_t)A_ML * sizeof(double2) +
           (size_t)((ntile + 3) & ~3) * sizeof(int) + 16;
}
static size_t synthesis_smem() { return (size_t)S_STAGES * S_STAGE_BYTES + 2 * S_STAGES * sizeof(uint64_t) + 4 * S_LC * sizeof(double2) + 64; }

cudaError_t launch_lambda_blocks(sht_plan_s* pl, const DevicePlan& d, bool analysis, cudaStream_t st)
{
    if (d.spin == 2) return launch_lambda_blocks_spin2(pl, d, analysis, st);
    if (!(pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam)) return cudaSuccess;
    if (analysis) {
        k_lambda_blocks_analysis<<<dim3((unsigned)(d.ntile_max * d.nck_max), (unsigned)(d.lmax + 1)), 128, 0, st>>>(d, pl->lam, pl->lam_i0);
        pl->launches++;
    } else if (d.nst_max > 0) {
        k_lambda_blocks_synthesis<<<dim3((unsigned)d.nst_max, (unsigned)d.npb, (unsigned)(d.lmax + 1)), 64, 0, st>>>(d, pl->lam);
        pl->launches++;
    }
    return cudaGetLastError();
}

// pstar > 0 (hybrid sweep of Alg. 3): only the ring chunks that start at or past ring pair pstar
// m_begin / m_count (spin 0): only the orders m_begin .. m_begin + m_count - 1 (m_count < 0: up to lmax)
cudaError_t launch_legendre_analysis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                     bool accumulate, cudaStream_t st, int pol, bool gen_lambda, int pstar, int m_begin, int m_count)
{
    if (d.spin == 2) return launch_legendre_analysis_spin2(pl, d, F, alm, k0, kmaps, accumulate, st, pol, gen_lambda, pstar);
    const int nm = m_count < 0 ? d.lmax + 1 - m_begin : m_count;
    if (nm <= 0) return cudaSuccess;
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    // leg_tsplit: one CTA per (m, l tile, k-tile) instead of per (m, k-tile): the l tiles of an (m, k-tile) then read the
    // same T_m boxes at about the same time from different SMs, and L2 serves the re-reads
    const int tsplit = pl->leg_tsplit;
    const int ntile0 = (d.lmax - m_begin) / A_ML + 1;      // the grid is sized for the tile groups of the first order
    const unsigned grid = (unsigned)(nm * nkt * (tsplit ? (ntile0 + tsplit - 1) / tsplit : 1));
    const size_t sm = analysis_smem(d.ntile_max);
    cudaError_t e = cudaFuncSetAttribute(k_legendre_analysis<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tmF;
    if ((e = make_tmap_F(d, F, KTILE_MAPS / KG, 1, &tmF)) != cudaSuccess) return e;
    const bool staged = pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam;
    if (staged && gen_lambda && (e = launch_lambda_blocks(pl, d, true, st)) != cudaSuccess) return e;
    k_legendre_analysis<0><<<grid, LEG_THREADS, sm, st>>>(tmF, d, alm, k0, kmaps, nkt, accumulate ? 1 : 0,
                                                       staged ? pl->lam : nullptr, staged ? pl->lam_i0 : nullptr, m_begin, tsplit, nullptr,
                                                       pstar, 0);
    pl->launches++;
    return cudaGetLastError();
}

// ---- one order m at a time (Alg. 3): the same kernels on the cells of order m only, lambda generated
// in the kernel (fused mode).  The tensor maps are built once per sweep by the caller.
cudaError_t legendre_order_maps(const DevicePlan& d, const double* F, const double* da, int kmaps, CUtensorMap* tmF, CUtensorMap* tmA)
{
    if (d.spin == 2) return legendre_order_maps_spin2(d, F, da, kmaps, tmF, tmA);
    cudaError_t e = cudaFuncSetAttribute(k_legendre_analysis<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)analysis_smem(d.ntile_max));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_legendre_analysis<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)analysis_smem(d.ntile_max));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_legendre_synthesis<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)synthesis_smem());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_legendre_synthesis<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)synthesis_smem());
    if (e == cudaSuccess) e = make_tmap_F(d, F, KTILE_MAPS / KG, 1, tmF);
    if (e == cudaSuccess) e = make_tmap_alm(d, da, (long long)kmaps * d.ncomp, tmA);
    return e;
}

// alm (rows from k0) += analysis of the orders m .. m + nm - 1 of F; da (rows from 0) = that increment
// pstar > 0 (hybrid sweep): only the ring chunks before the first one at or past pstar, and da holds the part of the
// increment that the later chunks give (launch_legendre_analysis with the same pstar): it is added and da completed
cudaError_t launch_legendre_analysis_order(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmF, double* alm, double* da,
                                           int k0, int kmaps, int m, int nm, cudaStream_t st, int pstar)
{
    if (d.spin == 2) return launch_legendre_analysis_order_spin2(pl, d, tmF, alm, da, k0, kmaps, m, nm, st, pstar);
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    const int ntile = (d.lmax - m) / A_ML + 1;
    // windowed (four CTAs per l tile) while the launch would not fill the SMs once: a per-order launch is a link in a chain
    // of dependent launches, so what counts is the serial work of one CTA (nside 128: 8 - 24 CTAs; 57 -> 24 ms per call);
    // past one wave the windows only multiply the operand reads (nside 512, 512 maps: 900 ms unwindowed, 979 ms windowed)
    if (nm * ntile * nkt <= pl->sm_count)
        k_legendre_analysis<1><<<(unsigned)(4 * nm * ntile * nkt), LEG_THREADS, analysis_smem(d.ntile_max), st>>>(tmF, d, alm, k0, kmaps, nkt, 1, nullptr,
                                                                                                          nullptr, m, 1, da, pstar, pstar > 0 ? 1 : 0);
    else
        k_legendre_analysis<0><<<(unsigned)(nm * ntile * nkt), LEG_THREADS, analysis_smem(d.ntile_max), st>>>(tmF, d, alm, k0, kmaps, nkt, 1, nullptr,
                                                                                                      nullptr, m, 1, da, pstar, pstar > 0 ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

// F (north / south) at the orders m .. m + nm - 1 = synthesis of those orders of da (rows from 0)
// pbend > 0 (hybrid sweep): only the first pbend blocks of 64 ring pairs
cudaError_t launch_legendre_synthesis_order(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmA, double* F, int kmaps, int m,
                                            int nm, cudaStream_t st, int pbend)
{
    if (d.spin == 2) return launch_legendre_synthesis_order_spin2(pl, d, tmA, F, kmaps, m, nm, st, pbend);
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    const int npb = (d.nh + S_PB - 1) / S_PB;
    const int nb = pbend > 0 && pbend < npb ? pbend : npb;
    if (nm * nkt * nb <= pl->sm_count)       // windowed under the same rule as the per-order analysis launch
        k_legendre_synthesis<1><<<(unsigned)(4 * nm * nkt * nb), LEG_THREADS, synthesis_smem(), st>>>(tmA, d, F, 0, kmaps, nkt, npb, nullptr, m, nb, 0, nb);
    else
        k_legendre_synthesis<0><<<(unsigned)(nm * nkt * nb), LEG_THREADS, synthesis_smem(), st>>>(tmA, d, F, 0, kmaps, nkt, npb, nullptr, m, nb, 0, nb);
    pl->launches++;
    return cudaGetLastError();
}

// pb0 > 0 (hybrid sweep of Alg. 3): only the blocks of 64 ring pairs from block pb0 on
cudaError_t launch_legendre_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps, cudaStream_t st,
                                      int pol, bool gen_lambda, int pb0, int m_begin, int m_count)
{
    if (d.spin == 2) return launch_legendre_synthesis_spin2(pl, d, alm, F, k0, kmaps, st, pol, gen_lambda, pb0);
    const size_t sm = synthesis_smem();
    cudaError_t e = cudaFuncSetAttribute(k_legendre_synthesis<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    CUtensorMap tmA;
    if ((e = make_tmap_alm(d, alm, (long long)(k0 + kmaps) * d.ncomp, &tmA)) != cudaSuccess) return e;
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    const int npb = (d.nh + S_PB - 1) / S_PB;
    const bool staged = pl->lam_mode == SHT_LAMBDA_STAGED && pl->lam;
    if (staged && gen_lambda && (e = launch_lambda_blocks(pl, d, false, st)) != cudaSuccess) return e;
    // leg_nsplit CTAs share the ring blocks of an (m, k-tile) (block b goes to CTA b mod nsplit): they re-read the same
    // a_lm tile at about the same time, and the set in flight (148 / nsplit tiles of up to 1.5 MB) fits L2
    const int nsplit = pl->leg_nsplit < 1 ? 1 : (pl->leg_nsplit > npb - pb0 ? npb - pb0 : pl->leg_nsplit);
    const int nm = m_count < 0 ? d.lmax + 1 - m_begin : m_count;
    if (nm <= 0) return cudaSuccess;
    k_legendre_synthesis<0><<<nm * nkt * nsplit, LEG_THREADS, sm, st>>>(tmA, d, F, k0, kmaps, nkt, npb, staged ? pl->lam : nullptr, m_begin, nsplit,
                                                                     pb0, npb);
    pl->launches++;
    return cudaGetLastError();
}

}  // namespace sht
