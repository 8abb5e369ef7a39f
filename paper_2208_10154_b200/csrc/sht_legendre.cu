// sht_legendre.cu -- subsystem (2): fused Legendre recurrence + FP64 tensor-core (DMMA.8x8x4) contraction,
// and subsystem (3): the m-major a_lm scatter / gather in its prologue / epilogue.
//
//   analysis  (PAPER.md:56-60 eq. 3, :95 eq. 7):  A_m = P_m T_m, contraction over ring pairs p,
//       a_lm^k = sum_p lambda_lm(theta_p) X_p^k,  X = E (l+m even) or O (l+m odd)   [N/S fold]
//   synthesis (PAPER.md:74-76 eq. 5, :97 eq. 7):  T_m = P_m^t A_m, contraction over l,
//       Ee_p = sum_{l+m even} lambda_lm(theta_p) a_lm,  Oo_p likewise; north = Ee + Oo, south = Ee - Oo.
//
// lambda_lm tiles are produced on the fly by the three-term recurrence, started at the
// plan's l_safe(m,p) (item 11), written to shared memory and consumed as DMMA A fragments;
// rings whose lambda is below threshold for a whole tile are skipped (ring optimisation, item 10, :229).
#include "sht_internal.h"

namespace sht {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---- tile shapes ---------------------------------------------------------------------------------
constexpr int LEG_THREADS = 512;     // 16 warps as 4 (M) x 4 (N); each warp owns a 32 x 32 block of C
constexpr int A_ML = 128;            // analysis: l rows per tile (64 of each parity class)
constexpr int A_PC = 32;             // analysis: ring pairs per contraction chunk
constexpr int A_SX = NK + 4;         // X tile row stride (doubles), = 4 mod 16: conflict-free B fragments
constexpr int A_SL = A_PC + 2;       // lambda tile row stride, = 2 mod 8: conflict-free A fragments
constexpr int S_PB = 64;             // synthesis: ring pairs per tile (Ee rows + Oo rows = 128 C rows)
constexpr int S_LC = 32;             // synthesis: l values per contraction chunk (16 of each parity)
constexpr int S_SA = 2 * S_LC + 2;   // a_lm tile stride per map (doubles), = 2 mod 16
constexpr int S_SL = S_PB + 2;       // lambda tile row stride, = 2 mod 8

// ------------------------------------------------------------------------------------------------
// analysis kernel: one CTA per (m, k-tile); loops over l tiles (outer) and ring chunks (inner).
// ------------------------------------------------------------------------------------------------
struct AnalysisSmem {
    double X[2][A_PC][A_SX];         // E and O rows of the chunk
    double L[A_ML][A_SL];            // lambda[l - l0][p - pc]
    double2 coef[A_ML];              // (alpha, beta) of the tile's l values
};

__global__ void __launch_bounds__(LEG_THREADS, 1)
k_legendre_analysis(DevicePlan d, const double* __restrict__ F, double* __restrict__ alm, int k0, int kmaps,
                    int nkt, int accumulate)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    AnalysisSmem& S = *reinterpret_cast<AnalysisSmem*>(smem_raw);
    double* st1 = reinterpret_cast<double*>(smem_raw + sizeof(AnalysisSmem));   // lambda_{l-1} per ring
    double* st2 = st1 + d.nh;                                                    // lambda_{l-2}
    int* lsp = reinterpret_cast<int*>(st2 + d.nh);                               // l_safe per ring

    const int m = blockIdx.x / nkt, kt = blockIdx.x % nkt;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 2, wn = warp & 3;
    const int cls = wm >> 1;                         // 0: l - m even (uses E), 1: odd (uses O)
    const int rbase = (wm & 1) * 32;                 // first row of this warp inside its parity class
    const int lmax = d.lmax, nh = d.nh;
    const int comp = 0;

    for (int p = tid; p < nh; p += LEG_THREADS) {
        const double2 sd = d.seed[(size_t)m * nh + p];
        st1[p] = sd.x; st2[p] = sd.y;
        lsp[p] = d.lstart[(size_t)m * nh + p];
    }
    __syncthreads();
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    const double2* Fc = reinterpret_cast<const double2*>(F);

    for (int l0 = m; l0 <= lmax; l0 += A_ML) {
        // first ring that has any non-negligible lambda in this l tile (l_safe decreases towards the equator)
        int pstart;
        {
            int lo = 0, hi = nh;                     // first p with lsp[p] < l0 + A_ML
            while (lo < hi) { int mid = (lo + hi) >> 1; if (lsp[mid] < l0 + A_ML) hi = mid; else lo = mid + 1; }
            // rings with mlim[p] <= m were never written to the workspace (and have lambda = 0 throughout)
            int lo2 = 0, hi2 = nh;
            while (lo2 < hi2) { int mid = (lo2 + hi2) >> 1; if (d.mlim[mid] > m) hi2 = mid; else lo2 = mid + 1; }
            pstart = lo > lo2 ? lo : lo2;
        }
        if (tid < A_ML) {
            const int l = l0 + tid;
            S.coef[tid] = (l <= lmax) ? coefm[l] : make_double2(0.0, 0.0);
        }
        double c[4][4][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) { c[i][j][0] = 0.0; c[i][j][1] = 0.0; }

        for (int pc = pstart; pc < nh; pc += A_PC) {
            __syncthreads();                         // previous chunk consumed, coef visible
            // ---- X tile: rows pc .. pc+A_PC-1, E and O, 128 real columns of this k-tile
            for (int e = tid; e < 2 * A_PC * (NK / 2); e += LEG_THREADS) {
                const int col2 = e % (NK / 2);       // complex column
                const int r = (e / (NK / 2)) % A_PC;
                const int h = e / ((NK / 2) * A_PC);
                const int p = pc + r;
                double2 v = make_double2(0.0, 0.0);
                if (p < nh) {
                    const int k = kt * KTILE_MAPS + col2;
                    v = Fc[f_cell(d, p, k >> 2, m, comp, h) + (k & 3)];
                }
                *reinterpret_cast<double2*>(&S.X[h][r][2 * col2]) = v;
            }
            // ---- lambda tile: thread t < A_PC walks ring pc + t through the tile's l values
            if (tid < A_PC) {
                const int p = pc + tid;
                if (p < nh) {
                    double x1 = st1[p], x2 = st2[p];
                    const int ls = lsp[p];
                    const double z = d.z[p];
#pragma unroll 4
                    for (int r = 0; r < A_ML; ++r) {
                        const int l = l0 + r;
                        double v = 0.0;
                        if (l >= ls && l <= lmax) {
                            const double2 ab = S.coef[r];
                            v = fma(ab.x * z, x1, -(ab.y * x2));
                            x2 = x1; x1 = v;
                        }
                        S.L[r][tid] = v;
                    }
                    st1[p] = x1; st2[p] = x2;
                } else {
                    for (int r = 0; r < A_ML; ++r) S.L[r][tid] = 0.0;
                }
            }
            __syncthreads();
            // ---- DMMA: C[l, k'] += lambda[l, p] X[p, k']
#pragma unroll
            for (int ks = 0; ks < A_PC / 4; ++ks) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    a[i] = S.L[2 * (rbase + 8 * i + (lane >> 2)) + cls][4 * ks + (lane & 3)];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    b[j] = S.X[cls][4 * ks + (lane & 3)][wn * 32 + 8 * j + (lane >> 2)];
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
            }
        }
        // ---- epilogue: scatter to the m-major alm layout; a lane holds (re, im) of one (l, map)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int l = l0 + 2 * (rbase + 8 * i + (lane >> 2)) + cls;
            if (l > lmax) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int kk = kt * KTILE_MAPS + wn * 16 + 4 * j + (lane & 3);
                if (kk >= kmaps) continue;
                double2* dst = reinterpret_cast<double2*>(alm) +
                               ((size_t)(k0 + kk) * d.ncomp + comp) * d.nalm + ((long long)m * (2 * lmax + 1 - m) / 2) + l;
                double2 v = make_double2(c[i][j][0], m == 0 ? 0.0 : c[i][j][1]);
                if (accumulate) { const double2 o = *dst; v.x += o.x; v.y += o.y; }
                *dst = v;
            }
        }
        __syncthreads();                             // coef / L reuse by the next l tile
    }
}

// ------------------------------------------------------------------------------------------------
// synthesis kernel: one CTA per (m, ring block of 64, k-tile); loops over l chunks.
// ------------------------------------------------------------------------------------------------
struct SynthesisSmem {
    double A[KTILE_MAPS][S_SA];      // a_lm tile: [map][l - lc][re,im]
    double L[S_LC][S_SL];            // lambda[l - lc][p - pb]
    double2 coef[S_LC];
};

__global__ void __launch_bounds__(LEG_THREADS, 1)
k_legendre_synthesis(DevicePlan d, const double* __restrict__ alm, double* __restrict__ F, int k0, int kmaps,
                     int nkt, int npb)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SynthesisSmem& S = *reinterpret_cast<SynthesisSmem*>(smem_raw);
    double* Cs = reinterpret_cast<double*>(smem_raw);          // epilogue staging, reuses the mainloop smem

    // block order: m slowest (long m first), then ring block, k-tile fastest
    const int kt = blockIdx.x % nkt;
    const int pbi = (blockIdx.x / nkt) % npb;
    const int m = blockIdx.x / (nkt * npb);
    const int pb = pbi * S_PB;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 2, wn = warp & 3;
    const int cls = wm >> 1;
    const int rbase = (wm & 1) * 32;
    const int lmax = d.lmax, nh = d.nh;
    const int comp = 0;

    // per-ring recurrence state lives in registers of threads 0..S_PB-1
    double x1 = 0.0, x2 = 0.0, z = 0.0;
    int ls = lmax + 1;
    if (tid < S_PB && pb + tid < nh) {
        const double2 sd = d.seed[(size_t)m * nh + pb + tid];
        x1 = sd.x; x2 = sd.y; ls = d.lstart[(size_t)m * nh + pb + tid]; z = d.z[pb + tid];
    }
    // the ring of the block closest to the equator starts first (l_safe decreases with p)
    const int plast = min(pb + S_PB, nh) - 1;
    if (m >= d.mlim[plast]) return;                    // no ring of this block takes part in order m (never read)
    const int lfirst = d.lstart[(size_t)m * nh + plast];
    const double2* coefm = d.coef + ((long long)m * (2 * lmax + 1 - m) / 2);
    const double2* almc = reinterpret_cast<const double2*>(alm);

    double c[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { c[i][j][0] = 0.0; c[i][j][1] = 0.0; }

    // chunks are aligned to m so that (l - m) even <-> even local index
    const int cfirst = (lfirst > lmax) ? (lmax + 1) : m + ((lfirst - m) / S_LC) * S_LC;
    for (int lc = cfirst; lc <= lmax; lc += S_LC) {
        __syncthreads();
        if (tid < S_LC) {
            const int l = lc + tid;
            S.coef[tid] = (l <= lmax) ? coefm[l] : make_double2(0.0, 0.0);
        }
        // ---- a_lm tile, straight from the m-major ABI layout (one contiguous run per map)
        for (int e = tid; e < KTILE_MAPS * S_LC; e += LEG_THREADS) {
            const int ll = e % S_LC, kk = e / S_LC;
            const int l = lc + ll, k = kt * KTILE_MAPS + kk;
            double2 v = make_double2(0.0, 0.0);
            if (l <= lmax && k < kmaps) {
                v = almc[((size_t)(k0 + k) * d.ncomp + comp) * d.nalm + ((long long)m * (2 * lmax + 1 - m) / 2) + l];
                if (m == 0) v.y = 0.0;
            }
            *reinterpret_cast<double2*>(&S.A[kk][2 * ll]) = v;
        }
        __syncthreads();                              // coef visible to the generator threads
        if (tid < S_PB) {
#pragma unroll 4
            for (int r = 0; r < S_LC; ++r) {
                const int l = lc + r;
                double v = 0.0;
                if (l >= ls && l <= lmax) {
                    const double2 ab = S.coef[r];
                    v = fma(ab.x * z, x1, -(ab.y * x2));
                    x2 = x1; x1 = v;
                }
                S.L[r][tid] = v;
            }
        }
        __syncthreads();
        // ---- DMMA: C[p, k'] += lambda[l, p] a[l, k'] over the chunk's l of this warp's parity class
#pragma unroll
        for (int ks = 0; ks < S_LC / 8; ++ks) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i)
                a[i] = S.L[2 * (4 * ks + (lane & 3)) + cls][rbase + 8 * i + (lane >> 2)];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int n = wn * 32 + 8 * j + (lane >> 2);          // real column: map n/2, part n&1
                b[j] = S.A[n >> 1][2 * (2 * (4 * ks + (lane & 3)) + cls) + (n & 1)];
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(c[i][j][0], c[i][j][1], a[i], b[j]);
        }
    }
    // ---- epilogue: exchange Ee / Oo through smem, write north = Ee + Oo, south = Ee - Oo rows
    __syncthreads();
    constexpr int SC = NK + 4;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int row = cls * S_PB + rbase + 8 * i + (lane >> 2);
            const int col = wn * 32 + 8 * j + 2 * (lane & 3);
            *reinterpret_cast<double2*>(&Cs[row * SC + col]) = make_double2(c[i][j][0], c[i][j][1]);
        }
    __syncthreads();
    double2* Fc = reinterpret_cast<double2*>(F);
    for (int e = tid; e < S_PB * (NK / 2); e += LEG_THREADS) {
        const int col2 = e % (NK / 2), r = e / (NK / 2);
        const int p = pb + r;
        if (p >= nh) continue;
        const double2 ee = *reinterpret_cast<const double2*>(&Cs[r * SC + 2 * col2]);
        const double2 oo = *reinterpret_cast<const double2*>(&Cs[(S_PB + r) * SC + 2 * col2]);
        const int k = kt * KTILE_MAPS + col2;
        double2* dst = Fc + f_cell(d, p, k >> 2, m, comp, 0) + (k & 3);
        dst[0] = make_double2(ee.x + oo.x, ee.y + oo.y);
        dst[KG] = make_double2(ee.x - oo.x, ee.y - oo.y);
    }
}

static size_t analysis_smem(int nh) { return sizeof(AnalysisSmem) + (size_t)nh * (2 * sizeof(double) + sizeof(int)); }
static size_t synthesis_smem()
{
    size_t a = sizeof(SynthesisSmem), b = (size_t)2 * S_PB * (NK + 4) * sizeof(double);
    return a > b ? a : b;
}

cudaError_t launch_legendre_analysis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                     bool accumulate, cudaStream_t st)
{
    const size_t sm = analysis_smem(d.nh);
    cudaError_t e = cudaFuncSetAttribute(k_legendre_analysis, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    k_legendre_analysis<<<(d.lmax + 1) * nkt, LEG_THREADS, sm, st>>>(d, F, alm, k0, kmaps, nkt, accumulate ? 1 : 0);
    pl->launches++;
    return cudaGetLastError();
}

cudaError_t launch_legendre_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps, cudaStream_t st)
{
    const size_t sm = synthesis_smem();
    cudaError_t e = cudaFuncSetAttribute(k_legendre_synthesis, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    const int nkt = (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;
    const int npb = (d.nh + S_PB - 1) / S_PB;
    k_legendre_synthesis<<<(d.lmax + 1) * nkt * npb, LEG_THREADS, sm, st>>>(d, alm, F, k0, kmaps, nkt, npb);
    pl->launches++;
    return cudaGetLastError();
}

}  // namespace sht
