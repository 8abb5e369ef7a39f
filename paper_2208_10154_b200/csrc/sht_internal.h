// sht_internal.h -- plan structure and kernel launchers of the B200 batched-SHT library (not installed).
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include "../../include/sht.h"

namespace sht {

// ---- tile constants shared by the ring-FFT and Legendre kernels --------------------------------
constexpr int KTILE_MAPS = 64;               // maps per Legendre k-tile
constexpr int NK = 2 * KTILE_MAPS;           // real columns per k-tile (re,im interleaved)
constexpr int MAX_RADIX_LIST = 16;           // factors of one ring length

// One folded ring pair p = 0 .. nh-1: north ring i = p+1 and its mirror 4 nside - i (PAPER.md:211 grid;
// north_star: "ring pairs symmetric about the equator folded").  The equator (p = nh-1) has no partner.
struct RingPair {
    int n;                 // pixels in the ring (4 i in the caps, 4 nside in the belt)
    int shift;             // phi0 = shift * pi / n   (shift in {0,1})
    long long start_n;     // first pixel of the north ring
    long long start_s;     // first pixel of the south ring, -1 for the equator
    int tw_off;            // offset (double2 units) of this ring length's table W_{2n}[j] = exp(-i pi j / n)
    int fac_off;           // offset into the radix list
    int nfac;              // number of radix passes
    int kt;                // maps per CTA of the ring-FFT kernels for this ring length
    // Bluestein (chirp-z) for ring lengths with a large prime factor: nb = 0 means plain mixed radix
    int nb;                // power-of-two convolution length >= 2n-1 (0 if unused)
    int chirp_off;         // offset (double2) of chirp[j] = exp(-i pi j^2 / n), j = 0..n-1
    int bfilt_off;         // offset (double2) of FFT_nb(conj-chirp filter) / nb
    int btw_off;           // offset (double2) of W_{nb}[j] = exp(-2 pi i j / nb), j = 0..nb-1
};

struct DevicePlan {
    int nside, lmax, spin, ncomp, nh;
    long long npix, nalm;
    int kpad;                       // complex columns per workspace row (multiple of KTILE_MAPS)
    const RingPair* rings;          // [nh]
    const double* z;                // [nh] cos(theta_p)
    const double* sin2;             // [nh] sin^2(theta_p)
    const double2* tw;              // all twiddle tables
    const int* radix;               // all radix lists
    const double2* coef;            // [nalm] (alpha_lm, beta_lm), m-major like alm
    const int* lstart;              // [lmax+1][nh] l_safe(m, p)
    const double2* seed;            // [lmax+1][nh] (lambda_{ls-1}, lambda_{ls-2})
    const double2* spin2c;          // [lmax+1] per-l constants for spin 2 (unused for spin 0)
};

}  // namespace sht

struct sht_plan_s {
    sht::DevicePlan d;
    int nmaps;
    int chunk;                      // maps per internal chunk
    double* F;                      // workspace [nh][lmax+1][ncomp][2][kpad][2]
    size_t F_bytes;
    size_t table_bytes;
    void* dev_allocs[24];
    int n_allocs;
    int max_ring;                   // largest ring length
    int ring_kt_min;                // maps per ring-kernel CTA at the largest ring length
    size_t fft_smem;                // dynamic smem of the ring kernels
    int sm_count;
    long long launches;
    char err[512];
    // host-entry staging (allocated on first use)
    double* stage_maps[2];
    double* stage_alm[2];
    int host_kpad;                  // workspace columns per row in the host path (two chunks share F)
    int host_chunk;
    cudaStream_t hstream[2];
    bool host_ready;
    // optional per-stage timing (sht_plan_set_timing)
    bool timing;
    int n_ev;
    cudaEvent_t ev0[256], ev1[256];
    int ev_stage[256];
};

namespace sht {

// ring FFT stage (sht_ring_fft.cu)
cudaError_t launch_ring_analysis(sht_plan_s* pl, const DevicePlan& d, const double* maps, double* F, int k0, int kmaps, cudaStream_t st);
// maps of the chunk are maps[k0 .. k0+kmaps); if sub_from != nullptr the output is sub_from[ksub0 + k] - synthesis
cudaError_t launch_ring_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* maps, int k0, int kmaps,
                                  const double* sub_from, int ksub0, cudaStream_t st);
// Legendre stage (sht_legendre.cu)
cudaError_t launch_legendre_analysis(sht_plan_s* pl, const DevicePlan& d, const double* F, double* alm, int k0, int kmaps,
                                     bool accumulate, cudaStream_t st);
cudaError_t launch_legendre_synthesis(sht_plan_s* pl, const DevicePlan& d, const double* alm, double* F, int k0, int kmaps, cudaStream_t st);
// plan-time seed table (sht_plan.cu)
cudaError_t launch_seed_table(const DevicePlan& d, const double* cm, int* lstart, double2* seed, cudaStream_t st);
size_t ring_fft_smem_bytes(int max_ring, int kt);

}  // namespace sht
