// sht_internal.h -- plan structure and kernel launchers of the B200 batched-SHT library (not installed).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include "../../include/sht.h"

namespace sht {

// ---- constants shared by the ring-FFT and Legendre kernels ------------------------------------------
constexpr int KG = 4;                        // maps per workspace group (one 128-byte line = E|O of 4 maps)
constexpr int KTILE_MAPS = 64;               // maps per Legendre k-tile (spin 0); spin 2: 32 (Q,U) pairs
constexpr int NK = 2 * KTILE_MAPS;           // real columns per k-tile (re,im interleaved)
constexpr int LEG_A_ML = 128;                // l rows per tile of the Legendre analysis kernel
constexpr int LEG_CS = 16;                   // l granularity of the plan's recurrence-state table
constexpr int MAX_RADIX_LIST = 16;           // factors of one ring length
constexpr int RING_THREADS = 256;            // threads per CTA of the ring kernels (two CTAs per SM)
constexpr int RING_EMAX = 8192;              // most complex elements (ring length x maps) one ring CTA holds in smem
constexpr int BLUESTEIN_MIN_PRIME = 37;      // smallest prime factor of a ring length that switches to Bluestein
constexpr int RING_NCLASS = 4;               // launch classes of the ring kernels (by dynamic smem size)
// default grid shapes of the spin-0 Legendre kernels (SHT_OPT_LEG_TILES_PER_CTA, SHT_OPT_LEG_RING_SPLIT)
constexpr int LEG_TSPLIT_DEFAULT = 2, LEG_NSPLIT_DEFAULT = 3;

// One folded ring pair p = 0 .. nh-1: north ring i = p+1 and its mirror 4 nside - i (PAPER.md:211 grid;
// north_star: "ring pairs symmetric about the equator folded").  The equator (p = nh-1) has no partner.
struct RingPair {
    int n;                 // pixels in the ring (4 i in the caps, 4 nside in the belt)
    int shift;             // phi0 = shift * pi / n   (shift in {0,1})
    long long start_n;     // first pixel of the north ring
    long long start_s;     // first pixel of the south ring, -1 for the equator
    int tw_off;            // offset (double2 units) of this ring length's table W_{2n}[j] = exp(-i pi j / n)
    int fac_off;           // offset into the radix list (forward order; the inverse transform runs it backwards)
    int nfac;              // number of radix passes
    int kt;                // maps per CTA of the ring kernels for this ring length (power of two <= 16)
    int oop;               // 1: the radix list has a second generic (prime >= 11) pass, done out of place
    int mlim;              // only m < mlim are needed from / for this ring (ring optimisation)
    int perm_off;          // offset of this ring length's table perm[bin] = position after the forward transform
    // Bluestein (chirp-z) rings: ring lengths with a prime factor > BLUESTEIN_MIN_PRIME are transformed as a
    // circular convolution of length lc >= 2 n - 1, lc = 2^a, 3 2^a or 5 2^a (lc = 0: plain mixed radix)
    int lc;
    int b_tw_off;          // offset (double2) of W_{2 lc}[j] = exp(-i pi j / lc)
    int b_fac_off, b_nfac; // radix list of the length-lc transform (4s and a 2)
    int hf_off;            // offset (double2) of FFT_lc(conj chirp) / lc in forward-output position order; the chirp
                           // c_j, j < n, follows at hf_off + lc
    int psh;               // shared-memory padding: one element every 2^psh (power-of-two transforms), 31 = none
    int nbuf;              // elements per map of one transform buffer, padding included
    // power-of-two rings: the digit reversal is a bit permutation, computed instead of read from the table:
    // r = brev(k) >> (32 - pbits); pos = ((r & pm_hi) >> 1) | ((r & pm_lo) << 1) | (r & pm_keep);  pbits = 0: use the table
    int pbits;
    unsigned pm_hi, pm_lo, pm_keep;
    // chirp-z fast path of the cap rings (sht_ring_pow2.cu): convolution length (0: not on that path) and the offset
    // (double2) of [filter spectrum FFT_L(conj chirp) / L in natural order: cz_len][chirp c_j: n]
    int cz_len, cz_off;
    // mixed-radix fast path (sht_ring_mixed.cu): n = mr_r1 mr_r2 mr_r3, all >= 2 (mr_r1 = 0: not on that path)
    int mr_r1, mr_r2, mr_r3;
};

struct DevicePlan {
    int nside, lmax, spin, ncomp, nh;
    long long npix, nalm;
    int kpad;                       // map slots per workspace row (multiple of KTILE_MAPS)
    int nkg;                        // kpad / KG
    const RingPair* rings;          // [nh]
    const double* z;                // [nh] cos(theta_p)
    const double* sin2;             // [nh] sin^2(theta_p)
    const double2* tw;              // all twiddle tables
    const int* radix;               // all radix lists
    const unsigned short* perm;     // all digit-reversal tables (bin -> position in the transformed buffer)
    const double2* coef;            // [nalm] (alpha_lm, beta_lm), m-major like alm
    const int* lstart;              // [lmax+1][nh] l_safe(m, p)
    const double2* seed;            // [lmax+1][nh] (lambda_{ls-1}, lambda_{ls-2})
    // recurrence state (lambda_{b-1}, lambda_{b-2}) at every LEG_CS-th l of every order, b = m + LEG_CS c, exactly as the
    // running recurrence from l_safe would hold it (the start seed while b <= l_safe): lets several generator warps
    // work on different l ranges of one ring at the same time.  Index (csoff[m] + c) * nh + p.
    const double2* cseed;
    const long long* csoff;         // [lmax+2] chunks before order m
    const double2* spin2c;          // [lmax+1] per-l constants for spin 2 (unused for spin 0)
    const int* mlim;                // [nh] copy of RingPair::mlim (monotone non-decreasing in p)
    const int* pst;                 // [lmax+1][ntile_max] first ring pair that takes part in l tile t of order m
    int ntile_max;                  // l tiles of order 0
    // staged-lambda mode (spin 0): lambda tiles are written by a generator kernel to a scratch in HBM, block by block in
    // the order the contraction kernels consume them, and fetched with one bulk copy per stage
    const int* ablk_off;            // [lmax+1][ntile_max] first analysis block (32 rings x 128 l) of (m, l tile)
    const int* sblk_off;            // [lmax+1][npb] first synthesis block (32 l x 64 rings) of (m, ring block)
    const int* scfirst;             // [lmax+1][npb] first l of the first synthesis block (lmax + 1: none)
    const int* sminls8;             // [lmax+1][npb][8] smallest l_safe of every 8 ring pairs of a synthesis ring block
    int npb;                        // ring blocks of 64
    int nck_max, nst_max;           // most analysis chunks per (m, tile), most synthesis stages per (m, ring block)
};

// Workspace F (both directions): T_m^k(theta) of PAPER.md:52 for one chunk of maps,
//   F[p][kg][m][comp][h][kk][re,im]   doubles,   kg = k / KG, kk = k % KG,
// h = 0/1 = E/O (north+south, north-south) on the analysis side, north/south on the synthesis side.
// One (p, kg, m, comp) cell is a 128-byte line.  Returns the double2 index of (.., h, kk = 0).
__host__ __device__ __forceinline__ size_t f_cell(const DevicePlan& d, int p, int kg, int m, int comp, int h)
{
    return (((((size_t)p * d.nkg + kg) * (size_t)(d.lmax + 1) + m) * d.ncomp + comp) * 2 + h) * KG;
}

}  // namespace sht

struct sht_plan_s {
    sht::DevicePlan d;
    int nmaps;
    int chunk;                      // maps per internal chunk
    double* F;                      // workspace, layout above
    size_t F_bytes;
    size_t table_bytes;
    void* dev_allocs[64];
    int n_allocs;
    // ring-kernel launch classes: rings grouped by the dynamic shared memory their CTA needs
    int* class_rings[sht::RING_NCLASS];     // device lists of ring-pair indices
    int class_count[sht::RING_NCLASS];
    int class_ktmin[sht::RING_NCLASS];      // smallest kt in the class (decides grid.x)
    size_t class_smem[sht::RING_NCLASS];
    // belt fast path (sht_ring_pow2.cu): ring pairs belt_first .. belt_first + belt_count - 1 have length 2^belt_logn
    // (belt_logn = 0: none); class_*_nb are the launch classes of the general kernels without those pairs
    int belt_logn, belt_first, belt_count;
    int leg_tsplit, leg_nsplit;     // grid shapes of the spin-0 Legendre kernels (sht_legendre.cu launchers)
    bool gs_plain;                        // SHT_OPT_ITER_HYBRID = 0: always the plain sweep
    int gs2_pstar, gs2_msplit;            // two-phase hybrid sweep (2 nside <= lmax < 4 nside): the belt ring pairs from gs2_pstar on couple an
                                          // order m only with 4 nside - m, so the orders below / from gs2_msplit = 2 nside are two batches; 0: n/a
    int gs_pstar, gs_mcut;                // Alg. 3 hybrid sweep: ring pairs >= gs_pstar (a multiple of 64) are alias-free; orders >= gs_mcut
                                          // (even) touch no ring pair below gs_pstar.  gs_pstar = nh: no alias-free tail, plain sweep
    bool fast_ring;                 // SHT_OPT_RING_PATH: the belt / mixed-radix / chirp-z ring kernels are in use
    int* class_rings_nb[sht::RING_NCLASS];
    int class_count_nb[sht::RING_NCLASS];
    int class_ktmin_nb[sht::RING_NCLASS];
    // mixed-radix fast path: ring pairs by length class (MR_NCLASS), the longest ring of each class
    int* mr_rings[6];
    int mr_count[6], mr_nmax[6];
    // chirp-z fast path: ring pairs by convolution length (CZ_NCLASS compiled lengths), their W_L tables
    int* cz_rings[8];
    int cz_count[8], cz_tw_off[8];
    int sm_count;
    long long launches;
    double* Fmap;                   // Alg. 2: folded T_m of the input maps (allocated on the first iterative call)
    double* upow;                   // Alg. 2: [nh][ncomp][kpad] uncovered ring power
    bool iter_reserve_failed;       // the second workspace did not fit: Alg. 2 forms residual maps instead
    int iter_mode;                  // SHT_ITER_TM (default) / SHT_ITER_PIXEL / SHT_ITER_IMMEDIATE
    double* lam;                    // staged-lambda scratch (nullptr: fused generation inside the contraction kernels)
    size_t lam_bytes;
    int* lam_i0;                    // [analysis blocks] first 16-row block with a started recurrence
    int lam_mode;                   // SHT_LAMBDA_FUSED / SHT_LAMBDA_STAGED
    long long n_ablk, n_sblk;
    double exec_flops_tile[2];      // DMMA flops one k-tile executes (0 analysis, 1 synthesis; spin 0; -1 = not counted)
    bool ring_attr_set, resid_attr_set;   // dynamic shared-memory attributes of the ring kernels set on this plan's device
    char err[512];
    // host-entry staging (allocated on first use)
    double* stage_maps[4];
    double* stage_alm[4];
    float* stage_maps_f32[4];       // single-precision staging of the *_host_f32 entries (allocated on their first call)
    float* stage_alm_f32[4];
    bool host_f32_ready;
    int host_kpad;                  // workspace columns per row in the host path (host_nb chunks share F)
    int host_nb;                    // chunks in flight in the host path (streams, staging buffers, workspace slices)
    int host_chunk;
    cudaStream_t hstream[4];
    cudaStream_t cap_stream;        // Alg. 3: the sweep is captured on this stream (created on first use)
    cudaEvent_t hevent;             // host path: lambda blocks of the call are ready
    bool host_ready;
    // optional per-stage timing (sht_plan_set_timing)
    bool timing;
    int n_ev, cap_ev;               // brackets recorded since the last sht_plan_stage_ms / allocated slots (grown on demand)
    long long ev_dropped;           // brackets lost because a slot could not be allocated (reported by sht_plan_stage_ms)
    cudaEvent_t *ev0, *ev1;
    int* ev_stage;
};

namespace sht {

// ring FFT stage (sht_ring_fft.cu)
// upow (may be null): [nh][ncomp][kpad], += power of each ring pair in the bins no stored order reaches (Alg. 2 rms)
cudaError_t launch_ring_analysis(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st,
                                 double* upow = nullptr);
cudaError_t launch_ring_residual(sht_plan_s* pl, const DevicePlan& d, double* F, const double* Fmap, const double* upow, double* acc,
                                 int kmaps, cudaStream_t st);
// maps of the chunk are maps[k0 .. k0+kmaps); if sub_from != nullptr the output is sub_from[ksub0 + k] - synthesis
cudaError_t launch_ring_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps,
                                  const double* sub_from, int ksub0, cudaStream_t st);
// belt fast path (sht_ring_pow2.cu)
cudaError_t launch_ring_analysis_belt(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st);
cudaError_t launch_ring_synthesis_belt(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st);
// mixed-radix fast path of the cap rings (sht_ring_mixed.cu): length classes N <= 512, <= 1024, <= 2048
constexpr int MR_NCLASS = 3;
constexpr int MR_MIN_N = 256, MR_MAX_N = 2048;
cudaError_t launch_ring_analysis_mr(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st);
cudaError_t launch_ring_synthesis_mr(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st);
// chirp-z fast path of the cap rings: the compiled convolution lengths
constexpr int CZ_NCLASS = 7;
constexpr int CZ_LEN[CZ_NCLASS] = {512, 768, 1024, 1536, 2048, 3072, 4096};
constexpr int CZ_MIN_N = 132;                // shorter rings stay with the general kernels
cudaError_t launch_ring_analysis_cz(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st);
cudaError_t launch_ring_synthesis_cz(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps, cudaStream_t st);
// Legendre stage (sht_legendre.cu)
// pol: spin 2 only, 0 = E and B, SHT_POL_E / SHT_POL_B = that component alone (`alm` then holds one component);
// gen_lambda = false: staged mode, the lambda scratch already holds this direction's blocks (host path: one generator
// pass per call instead of one per chunk)
cudaError_t launch_legendre_analysis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                     bool accumulate, cudaStream_t st, int pol = 0, bool gen_lambda = true, int pstar = 0,
                                     int m_begin = 0, int m_count = -1);      // order range: spin 0 only
cudaError_t launch_legendre_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps, cudaStream_t st,
                                      int pol = 0, bool gen_lambda = true, int pb0 = 0, int m_begin = 0, int m_count = -1);
// the lambda-block generator kernel of the staged mode on its own (no-op in fused mode)
cudaError_t launch_lambda_blocks(sht_plan_s* pl, const DevicePlan& d, bool analysis, cudaStream_t st);
// Alg. 3, the orders m .. m + nm - 1 at a time: tensor maps once per chunk, then per step analysis (alm += , da =
// increment), synthesis of the increment into the cells of these orders of S, and the update of the residual workspace R
cudaError_t legendre_order_maps(const DevicePlan& d, const double* F, const double* da, int kmaps, CUtensorMap* tmF, CUtensorMap* tmA);
cudaError_t launch_legendre_analysis_order(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmF, double* alm, double* da,
                                           int k0, int kmaps, int m, int nm, cudaStream_t st, int pstar = 0);
cudaError_t launch_legendre_synthesis_order(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmA, double* F, int kmaps, int m,
                                            int nm, cudaStream_t st, int pbend = 0);
// np > 0: only the ring pairs p < np
cudaError_t launch_gs_update(sht_plan_s* pl, const DevicePlan& d, const double* S, double* R, int m, int nm, int kmaps, cudaStream_t st, int np = 0,
                             int p0 = 0);     // ring pairs p0 <= p < np
// hybrid sweep of Alg. 3 (sht_api.cu): the ring pairs from pstar on are alias-free (no two orders below their mlim share a
// bin), so all their orders are corrected in one launch: R -= re-expansion of S at every order, ring pairs >= pstar
cudaError_t launch_gs_update_free(sht_plan_s* pl, const DevicePlan& d, const double* S, double* R, int pstar, int kmaps, cudaStream_t st);
// alm (rows from k0) += da (rows from 0) at the orders m >= m0
cudaError_t launch_alm_add_from(sht_plan_s* pl, const DevicePlan& d, double* alm, const double* da, int k0, int kmaps, int m0, cudaStream_t st);
cudaError_t launch_ring_power(sht_plan_s* pl, const DevicePlan& d, const double* R, const double* upow, double* acc, int kmaps, cudaStream_t st);
constexpr size_t LAM_ABLK_BYTES = 2 * 32 * 66 * 8;      // one analysis lambda block: [class][32 rings][66] doubles
constexpr size_t LAM_SBLK_BYTES = 32 * 66 * 8;          // one synthesis lambda block: [32 l][66] doubles
// spin 2 (sht_legendre_spin2.cu); the spin-0 launchers dispatch to these
cudaError_t launch_legendre_analysis_spin2(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                           bool accumulate, cudaStream_t st, int pol, bool gen_lambda, int pstar);
cudaError_t launch_legendre_synthesis_spin2(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps,
                                            cudaStream_t st, int pol, bool gen_lambda, int pb0);
cudaError_t launch_lambda_blocks_spin2(sht_plan_s* pl, const DevicePlan& d, bool analysis, cudaStream_t st);
cudaError_t legendre_order_maps_spin2(const DevicePlan& d, const double* F, const double* da, int kmaps, CUtensorMap* tmF, CUtensorMap* tmA);
cudaError_t launch_legendre_analysis_order_spin2(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmF, double* alm, double* da,
                                                 int k0, int kmaps, int m, int nm, cudaStream_t st, int pstar);
cudaError_t launch_legendre_synthesis_order_spin2(sht_plan_s* pl, const DevicePlan& d, const CUtensorMap& tmA, double* F, int kmaps, int m,
                                                  int nm, cudaStream_t st, int pbend);
// plan-time seed table (sht_plan.cu)
cudaError_t launch_seed_table(const DevicePlan& d, const double* cm, int* lstart, double2* seed, cudaStream_t st);
cudaError_t launch_chunk_seeds(const DevicePlan& d, double2* cseed, cudaStream_t st);

}  // namespace sht
