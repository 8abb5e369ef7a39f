// sht_api.cu -- the C ABI of include/sht.h: argument checks, map chunking, stage sequencing.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include "sht_internal.h"
#include <nvtx3/nvToolsExt.h>       // header-only NVTX 3: ranges cost a pointer test when no tool is attached

using namespace sht;

namespace sht {

// sum of squares per (map, component) for the residual rms of Alg. 2 (reading G18 in DESIGN.md)
// rows = blockIdx.y + j * gridDim.y (the grid's y extent is capped at 65535)
__global__ void k_sumsq(const double* __restrict__ x, long long npix, int nrow, double* __restrict__ acc)
{
  for (int rowi = blockIdx.y; rowi < nrow; rowi += gridDim.y) {
    const double* row = x + (size_t)rowi * npix;
    double s = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < npix; i += (long long)gridDim.x * blockDim.x) {
        const double v = row[i];
        s = fma(v, v, s);
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ double ws[32];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = threadIdx.x < (blockDim.x >> 5) ? ws[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) atomicAdd(acc + rowi, s);
    }
    __syncthreads();
  }
}

__global__ void k_rms_finish(const double* __restrict__ acc, int n, double inv_npix, double* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = sqrt(acc[i] * inv_npix);
}

// eq. A7: all a_lm of one map in a real (lmax+1) x (lmax+1) square,
//   Re a_lm -> (l, m),   Im a_lm (m >= 1) -> (l - m, lmax - m + 1);   Im a_l0 is not stored (it is zero).
// One thread per a_lm slot of the m-major ABI layout.
template <bool PACK>
__global__ void k_a7(int lmax, long long nalm, long long rows, double* __restrict__ alm, double* __restrict__ sq)
{
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= rows * nalm) return;
    const long long row = gid / nalm;
    const long long idx = gid - row * nalm;
    // m from idx = m (2 lmax + 1 - m)/2 + l: largest m with offset(m) + m <= idx
    int m = (int)(((2.0 * lmax + 3.0) - sqrt((2.0 * lmax + 3.0) * (2.0 * lmax + 3.0) - 8.0 * (double)idx)) * 0.5);
    if (m < 0) m = 0;
    if (m > lmax) m = lmax;
    while (m > 0 && (long long)m * (2 * lmax + 1 - m) / 2 + m > idx) --m;
    while (m < lmax && (long long)(m + 1) * (2 * lmax - m) / 2 + (m + 1) <= idx) ++m;
    const int l = (int)(idx - (long long)m * (2 * lmax + 1 - m) / 2);
    const long long n1 = lmax + 1;
    double* s = sq + row * n1 * n1;
    double2* a = reinterpret_cast<double2*>(alm) + gid;
    if (PACK) {
        const double2 v = *a;
        s[(long long)l * n1 + m] = v.x;
        if (m >= 1) s[(long long)(l - m) * n1 + (lmax - m + 1)] = v.y;
    } else {
        *a = make_double2(s[(long long)l * n1 + m], m >= 1 ? s[(long long)(l - m) * n1 + (lmax - m + 1)] : 0.0);
    }
}

// register-resident DMMA loop for the roofline denominator
__global__ void k_mma_peak(double* out, int iters)
{
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace sht

static sht_status_t cuda_fail(sht_plan_t pl, const char* what, cudaError_t e)
{
    snprintf(pl->err, sizeof(pl->err), "%s: %s", what, cudaGetErrorString(e));
    return SHT_ERR_CUDA;
}

#define SHT_TRY(call, what)                                   \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(pl, what, e__); \
    } while (0)

// stream-ordered scratch that is released on every exit path (SHT_TRY returns early)
struct AsyncScratch {
    void* p = nullptr;
    cudaStream_t st;
    explicit AsyncScratch(cudaStream_t s) : st(s) {}
    AsyncScratch(const AsyncScratch&) = delete;
    AsyncScratch& operator=(const AsyncScratch&) = delete;
    ~AsyncScratch() { if (p) cudaFreeAsync(p, st); }
    cudaError_t alloc(size_t bytes) { return cudaMallocAsync(&p, bytes ? bytes : 16, st); }
    double* d() const { return static_cast<double*>(p); }
};

// NVTX range around the launches of one stage / one entry (host-side: it brackets the enqueue, which is what a timeline
// tool attributes the kernels launched inside to)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange&) = delete;
    NvtxRange& operator=(const NvtxRange&) = delete;
};

// ---- optional per-stage timing ---------------------------------------------------------------------
static int timing_begin(sht_plan_t pl, int stage, cudaStream_t st)
{
    if (!pl->timing) return -1;
    if (pl->n_ev == pl->cap_ev) {                        // grow the event arrays (Alg. 3 records thousands of brackets)
        const int cap = pl->cap_ev ? 2 * pl->cap_ev : 256;
        cudaEvent_t* a = (cudaEvent_t*)realloc(pl->ev0, (size_t)cap * sizeof(cudaEvent_t));
        if (a) pl->ev0 = a;
        cudaEvent_t* b = a ? (cudaEvent_t*)realloc(pl->ev1, (size_t)cap * sizeof(cudaEvent_t)) : nullptr;
        if (b) pl->ev1 = b;
        int* c = b ? (int*)realloc(pl->ev_stage, (size_t)cap * sizeof(int)) : nullptr;
        if (c) pl->ev_stage = c;
        if (!a || !b || !c) { pl->ev_dropped++; return -1; }
        for (int i = pl->cap_ev; i < cap; ++i) { pl->ev0[i] = nullptr; pl->ev1[i] = nullptr; }
        pl->cap_ev = cap;
    }
    const int i = pl->n_ev;
    if (!pl->ev0[i] && (cudaEventCreate(&pl->ev0[i]) != cudaSuccess || cudaEventCreate(&pl->ev1[i]) != cudaSuccess)) {
        cudaGetLastError();
        pl->ev_dropped++;
        return -1;
    }
    pl->n_ev++;
    pl->ev_stage[i] = stage;
    cudaEventRecord(pl->ev0[i], st);
    return i;
}
static void timing_end(sht_plan_t pl, int i, cudaStream_t st)
{
    if (i >= 0) cudaEventRecord(pl->ev1[i], st);
}

extern "C" sht_status_t sht_plan_set_timing(sht_plan_t pl, int enable)
{
    if (!pl) return SHT_ERR_NULL;
    pl->timing = enable != 0;
    pl->n_ev = 0;
    pl->ev_dropped = 0;
    return SHT_OK;
}

extern "C" sht_status_t sht_plan_stage_ms(sht_plan_t pl, double* ms4, int* n4)
{
    if (!pl || !ms4 || !n4) return SHT_ERR_NULL;
    for (int s = 0; s < 4; ++s) { ms4[s] = 0.0; n4[s] = 0; }
    for (int i = 0; i < pl->n_ev; ++i) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(pl->ev1[i]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, pl->ev0[i], pl->ev1[i]);
        if (e != cudaSuccess) { snprintf(pl->err, sizeof(pl->err), "stage timing: %s", cudaGetErrorString(e)); return SHT_ERR_CUDA; }
        ms4[pl->ev_stage[i]] += t; n4[pl->ev_stage[i]]++;
    }
    pl->n_ev = 0;
    if (pl->ev_dropped) {                                // never silently: the sums would be short
        snprintf(pl->err, sizeof(pl->err), "stage timing: %lld brackets could not be recorded", pl->ev_dropped);
        pl->ev_dropped = 0;
        return SHT_ERR_ALLOC;
    }
    return SHT_OK;
}

// maps[kmap0 .. kmap0+kmaps) -> alm[kalm0 .. kalm0+kmaps)
static sht_status_t analysis_chunk(sht_plan_t pl, const DevicePlan& d, const double* maps, int kmap0, double* alm,
                                   int kalm0, double* F, int kmaps, bool accumulate, cudaStream_t st, int pol = 0,
                                   bool gen_lambda = true)
{
    int t = timing_begin(pl, 0, st);
    {
        NvtxRange r("sht: ring FFT + mapping (analysis)");
        SHT_TRY(launch_ring_analysis(pl, d, maps, F, kmap0, kmaps, st), "ring analysis");
    }
    timing_end(pl, t, st);
    t = timing_begin(pl, 1, st);
    {
        NvtxRange r("sht: Legendre analysis");
        SHT_TRY(launch_legendre_analysis(pl, d, F, alm, kalm0, kmaps, accumulate, st, pol, gen_lambda), "legendre analysis");
    }
    timing_end(pl, t, st);
    return SHT_OK;
}

// alm[kalm0 ..) -> maps[kmap0 ..); with sub_from: maps = sub_from[ksub0 ..] - synthesis
static sht_status_t synthesis_chunk(sht_plan_t pl, const DevicePlan& d, const double* alm, int kalm0, double* maps,
                                    int kmap0, double* F, int kmaps, const double* sub_from, int ksub0, cudaStream_t st,
                                    int pol = 0, bool gen_lambda = true)
{
    int t = timing_begin(pl, 2, st);
    {
        NvtxRange r("sht: Legendre synthesis");
        SHT_TRY(launch_legendre_synthesis(pl, d, alm, F, kalm0, kmaps, st, pol, gen_lambda), "legendre synthesis");
    }
    timing_end(pl, t, st);
    t = timing_begin(pl, 3, st);
    {
        NvtxRange r("sht: mapping + ring FFT (synthesis)");
        SHT_TRY(launch_ring_synthesis(pl, d, F, maps, kmap0, kmaps, sub_from, ksub0, st), "ring synthesis");
    }
    timing_end(pl, t, st);
    return SHT_OK;
}

extern "C" sht_status_t sht_analysis(sht_plan_t pl, const double* maps, double* alm, void* stream)
{
    NvtxRange nvtx_entry("sht_analysis");
    if (!pl) return SHT_ERR_NULL;
    if (!maps || !alm) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    cudaStream_t st = (cudaStream_t)stream;
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        sht_status_t s = analysis_chunk(pl, pl->d, maps, k0, alm, k0, pl->F, kmaps, false, st);
        if (s != SHT_OK) return s;
    }
    return SHT_OK;
}

extern "C" sht_status_t sht_synthesis(sht_plan_t pl, const double* alm, double* maps, void* stream)
{
    NvtxRange nvtx_entry("sht_synthesis");
    if (!pl) return SHT_ERR_NULL;
    if (!maps || !alm) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    cudaStream_t st = (cudaStream_t)stream;
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        sht_status_t s = synthesis_chunk(pl, pl->d, alm, k0, maps, k0, pl->F, kmaps, nullptr, 0, st);
        if (s != SHT_OK) return s;
    }
    return SHT_OK;
}

// E-only / B-only polarisation transforms (item 9)
static sht_status_t pol_run(sht_plan_t pl, const double* maps, const double* alm_in, double* maps_out, double* alm_out, int which,
                            void* stream)
{
    if (!pl) return SHT_ERR_NULL;
    if ((!maps && !maps_out) || (!alm_in && !alm_out)) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    if (pl->d.spin != 2 || (which != SHT_POL_E && which != SHT_POL_B)) {
        snprintf(pl->err, sizeof(pl->err), "E-only / B-only transforms need a spin-2 plan and which = SHT_POL_E or SHT_POL_B");
        return SHT_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    sht_status_t s = SHT_OK;
    for (int k0 = 0; k0 < pl->nmaps && s == SHT_OK; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        s = alm_out ? analysis_chunk(pl, pl->d, maps, k0, alm_out, k0, pl->F, kmaps, false, st, which)
                    : synthesis_chunk(pl, pl->d, alm_in, k0, maps_out, k0, pl->F, kmaps, nullptr, 0, st, which);
    }
    return s;
}

extern "C" sht_status_t sht_analysis_pol(sht_plan_t pl, const double* maps, double* alm, int which, void* stream)
{
    return pol_run(pl, maps, nullptr, nullptr, alm, which, stream);
}

extern "C" sht_status_t sht_synthesis_pol(sht_plan_t pl, const double* alm, double* maps, int which, void* stream)
{
    return pol_run(pl, nullptr, alm, maps, nullptr, which, stream);
}

// Alg. 2 kept between T_m and a_lm (item 8): one ring-FFT pass over the maps, then per round a Legendre
// synthesis, the residual on the ring spectra (k_ring_residual) and a Legendre analysis with accumulation.  Needs a
// second workspace (the folded T_m of the maps); if that does not fit, falls back to forming the residual maps.
static sht_status_t iter_tm_space(sht_plan_t pl, const double* maps, double* alm, int niter, double* resid_rms, cudaStream_t st)
{
    const DevicePlan& d = pl->d;
    AsyncScratch accs(st);
    SHT_TRY(accs.alloc((size_t)pl->chunk * d.ncomp * sizeof(double)), "rms scratch");
    double* acc = accs.d();
    const size_t ubytes = (size_t)d.nh * d.ncomp * d.kpad * sizeof(double);
    sht_status_t s = SHT_OK;
    for (int k0 = 0; k0 < pl->nmaps && s == SHT_OK; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        const int nrow = kmaps * d.ncomp;
        SHT_TRY(cudaMemsetAsync(pl->upow, 0, ubytes, st), "uncovered-power memset");
        int t = timing_begin(pl, 0, st);
        SHT_TRY(launch_ring_analysis(pl, d, maps, pl->Fmap, k0, kmaps, st, pl->upow), "ring analysis");
        timing_end(pl, t, st);
        t = timing_begin(pl, 1, st);
        SHT_TRY(launch_legendre_analysis(pl, d, pl->Fmap, alm, k0, kmaps, false, st), "legendre analysis");
        timing_end(pl, t, st);
        for (int it = 0; it < niter && s == SHT_OK; ++it) {
            t = timing_begin(pl, 2, st);
            SHT_TRY(launch_legendre_synthesis(pl, d, alm, pl->F, k0, kmaps, st), "legendre synthesis");
            timing_end(pl, t, st);
            SHT_TRY(cudaMemsetAsync(acc, 0, (size_t)nrow * sizeof(double), st), "rms memset");
            t = timing_begin(pl, 3, st);
            SHT_TRY(launch_ring_residual(pl, d, pl->F, pl->Fmap, pl->upow, acc, kmaps, st), "ring residual");
            timing_end(pl, t, st);
            if (resid_rms) {
                k_rms_finish<<<(nrow + 127) / 128, 128, 0, st>>>(acc, nrow, 1.0 / (double)d.npix,
                                                                 resid_rms + (size_t)it * pl->nmaps * d.ncomp + (size_t)k0 * d.ncomp);
                pl->launches++;
                SHT_TRY(cudaGetLastError(), "rms kernel");
            }
            t = timing_begin(pl, 1, st);
            SHT_TRY(launch_legendre_analysis(pl, d, pl->F, alm, k0, kmaps, true, st), "legendre analysis");
            timing_end(pl, t, st);
        }
    }
    return s;
}

// Alg. 3, the "immediate" iteration (reading G21 in DESIGN.md): a^0 by the plain analysis, the
// residual R = T_m(map) - alias(T_m(synthesis a^0)) for all orders, then niter sweeps over m = 0 .. lmax in this order:
// delta a_m = Legendre analysis of R at order m, a_m += delta a_m, Legendre synthesis of delta a_m at order m, and R
// corrected at every order that shares a ring bin with m -- so the orders that follow see the correction (Gauss-Seidel).
// Sequential in m within each parity class: 3 launches per pair of orders (m even, m + 1) and sweep.  Spin 0 and spin 2
// (E and B of an order are corrected together).
static sht_status_t iter_immediate(sht_plan_t pl, const double* maps, double* alm, int niter, double* resid_rms, cudaStream_t st)
{
    const DevicePlan& d = pl->d;
    AsyncScratch accs(st), das(st);
    SHT_TRY(accs.alloc((size_t)pl->chunk * d.ncomp * sizeof(double)), "rms scratch");
    SHT_TRY(das.alloc((size_t)pl->chunk * d.ncomp * d.nalm * 2 * sizeof(double)), "increment scratch");
    double* acc = accs.d(); double* da = das.d();
    const size_t ubytes = (size_t)d.nh * d.ncomp * d.kpad * sizeof(double);
    double* R = pl->F;              // residual, folded (even / odd), all orders
    double* S = pl->Fmap;           // T_m(map) first, then the synthesised increment of one order at a time
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        const int nrow = kmaps * d.ncomp;
        SHT_TRY(cudaMemsetAsync(pl->upow, 0, ubytes, st), "uncovered-power memset");
        int t = timing_begin(pl, 0, st);
        SHT_TRY(launch_ring_analysis(pl, d, maps, S, k0, kmaps, st, pl->upow), "ring analysis");
        timing_end(pl, t, st);
        t = timing_begin(pl, 1, st);
        SHT_TRY(launch_legendre_analysis(pl, d, S, alm, k0, kmaps, false, st), "legendre analysis");
        timing_end(pl, t, st);
        t = timing_begin(pl, 2, st);
        SHT_TRY(launch_legendre_synthesis(pl, d, alm, R, k0, kmaps, st), "legendre synthesis");
        timing_end(pl, t, st);
        SHT_TRY(cudaMemsetAsync(acc, 0, (size_t)nrow * sizeof(double), st), "rms memset");
        t = timing_begin(pl, 3, st);
        SHT_TRY(launch_ring_residual(pl, d, R, S, pl->upow, acc, kmaps, st), "ring residual");
        timing_end(pl, t, st);
        CUtensorMap tmF, tmA;
        SHT_TRY(legendre_order_maps(d, R, da, kmaps, &tmF, &tmA), "tensor maps");
        // One sweep is the same sequence of (lmax + 1) / 2 x 3 dependent launches for every iteration of the chunk: it is
        // captured once into a CUDA graph and replayed (launch overhead of ~9 k launches per sweep at config 5).  If the
        // caller's stream cannot be captured (it is itself under capture), the launches are issued directly.
        // an even and an odd order never fall on the same bin of a ring of 4q pixels (m' = +-m mod 4q keeps the parity):
        // the orders m, m + 1 of a step are independent, and the sweep equals the one-by-one sweep bit for bit
        // Hybrid sweep: the ring pairs from gs_pstar on are alias-free (sht_plan.cu), their orders never correct
        // one another, so what they give to delta a_m does not depend on the sweep's progress and what delta a_m gives
        // back to them is read by no later order of the sweep.  Their share of the analysis therefore runs first as ONE
        // whole-transform launch (-> da), the chain of dependent steps covers only the ring pairs below gs_pstar and the
        // orders below gs_mcut (delta a_m = da_m + their share; a_m += delta a_m; their R corrected at once), and the
        // alias-free ring pairs get the synthesis of the complete da and their correction as two launches at the end.
        // Equal to the one-by-one sweep up to the order of the ring sums.  Used when at least half of the ring pairs
        // are alias-free (lmax <= 2 nside: the paper's case for Alg. 3).
        const int pstar = pl->gs_pstar, mcut = pl->gs_mcut < d.lmax + 1 ? pl->gs_mcut : d.lmax + 1;
        const bool hybrid = !pl->gs_plain && pstar <= d.nh / 2;
        // Two-phase variant (2 nside <= lmax < 4 nside, spin 0): the belt ring pairs (from gs2_pstar on) are not alias-free,
        // but an order m meets only 4 nside - m there.  The orders below 2 nside never meet one another on the belt, nor do
        // the orders from 2 nside on: each of the two groups is handled like the alias-free case -- the belt's share of the
        // group's delta a first (one launch), the chain over the cap ring pairs, then the belt synthesis of the group
        // and its correction (every target order, also those of the other group) -- and the second group starts from
        // the belt residual the first one left.
        const int p2 = pl->gs2_pstar, msplit = pl->gs2_msplit;
        const bool twophase = !hybrid && !pl->gs_plain && d.spin == 0 && msplit > 0 && msplit <= d.lmax;
        auto sweep = [&](cudaStream_t ss) -> sht_status_t {
            if (twophase) {
                for (int ph = 0; ph < 2; ++ph) {
                    const int ma = ph ? msplit : 0, mb = ph ? d.lmax + 1 : msplit;      // msplit = 2 nside is even: pairs do not straddle
                    SHT_TRY(launch_legendre_analysis(pl, d, R, da, 0, kmaps, false, ss, 0, true, p2, ma, mb - ma), "legendre analysis (belt)");
                    for (int m = ma; m < mb; m += 2) {
                        const int nm = m + 1 < mb ? 2 : 1;
                        SHT_TRY(launch_legendre_analysis_order(pl, d, tmF, alm, da, k0, kmaps, m, nm, ss, p2), "legendre analysis (orders m, m+1)");
                        SHT_TRY(launch_legendre_synthesis_order(pl, d, tmA, S, kmaps, m, nm, ss, p2 / 64), "legendre synthesis (orders m, m+1)");
                        SHT_TRY(launch_gs_update(pl, d, S, R, m, nm, kmaps, ss, p2), "residual update");
                    }
                    SHT_TRY(launch_legendre_synthesis(pl, d, da, S, 0, kmaps, ss, 0, true, p2 / 64, ma, mb - ma), "legendre synthesis (belt)");
                    SHT_TRY(launch_gs_update(pl, d, S, R, ma, mb - ma, kmaps, ss, 0, p2), "residual update (belt)");
                }
                return SHT_OK;
            }
            if (hybrid) {
                SHT_TRY(launch_legendre_analysis(pl, d, R, da, 0, kmaps, false, ss, 0, true, pstar), "legendre analysis (alias-free ring pairs)");
                for (int m = 0; m < mcut; m += 2) {
                    const int nm = m < d.lmax ? 2 : 1;
                    SHT_TRY(launch_legendre_analysis_order(pl, d, tmF, alm, da, k0, kmaps, m, nm, ss, pstar), "legendre analysis (orders m, m+1)");
                    SHT_TRY(launch_legendre_synthesis_order(pl, d, tmA, S, kmaps, m, nm, ss, pstar / 64), "legendre synthesis (orders m, m+1)");
                    SHT_TRY(launch_gs_update(pl, d, S, R, m, nm, kmaps, ss, pstar), "residual update");
                }
                SHT_TRY(launch_alm_add_from(pl, d, alm, da, k0, kmaps, mcut, ss), "a_lm increment (orders >= gs_mcut)");
                SHT_TRY(launch_legendre_synthesis(pl, d, da, S, 0, kmaps, ss, 0, true, pstar / 64), "legendre synthesis (alias-free ring pairs)");
                SHT_TRY(launch_gs_update_free(pl, d, S, R, pstar, kmaps, ss), "residual update (alias-free ring pairs)");
                return SHT_OK;
            }
            for (int m = 0; m <= d.lmax; m += 2) {
                const int nm = m < d.lmax ? 2 : 1;
                SHT_TRY(launch_legendre_analysis_order(pl, d, tmF, alm, da, k0, kmaps, m, nm, ss), "legendre analysis (orders m, m+1)");
                SHT_TRY(launch_legendre_synthesis_order(pl, d, tmA, S, kmaps, m, nm, ss), "legendre synthesis (orders m, m+1)");
                SHT_TRY(launch_gs_update(pl, d, S, R, m, nm, kmaps, ss), "residual update");
            }
            return SHT_OK;
        };
        // captured on a stream of the plan's own (the legacy default stream cannot be captured), replayed on the caller's
        cudaGraphExec_t gexec = nullptr;
        long long sweep_launches = 0;
        if (niter > 0 && !pl->cap_stream && cudaStreamCreateWithFlags(&pl->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
            pl->cap_stream = nullptr;
            cudaGetLastError();
        }
        if (niter > 0 && pl->cap_stream && cudaStreamBeginCapture(pl->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const long long l0 = pl->launches;
            const sht_status_t cs = sweep(pl->cap_stream);
            sweep_launches = pl->launches - l0;
            pl->launches = l0;
            cudaGraph_t graph = nullptr;
            const cudaError_t ce = cudaStreamEndCapture(pl->cap_stream, &graph);
            if (cs != SHT_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) gexec = nullptr;
            if (graph) cudaGraphDestroy(graph);
            if (cs != SHT_OK) return cs;
        }
        cudaGetLastError();
        for (int it = 0; it < niter; ++it) {
            if (it > 0 && resid_rms) {
                SHT_TRY(cudaMemsetAsync(acc, 0, (size_t)nrow * sizeof(double), st), "rms memset");
                SHT_TRY(launch_ring_power(pl, d, R, pl->upow, acc, kmaps, st), "ring power");
            }
            if (resid_rms) {
                k_rms_finish<<<(nrow + 127) / 128, 128, 0, st>>>(acc, nrow, 1.0 / (double)d.npix,
                                                                 resid_rms + (size_t)it * pl->nmaps * d.ncomp + (size_t)k0 * d.ncomp);
                pl->launches++;
                SHT_TRY(cudaGetLastError(), "rms kernel");
            }
            t = timing_begin(pl, 1, st);
            if (gexec) {
                const cudaError_t ge = cudaGraphLaunch(gexec, st);
                if (ge != cudaSuccess) { cudaGraphExecDestroy(gexec); return cuda_fail(pl, "sweep graph launch", ge); }
                pl->launches += sweep_launches;
            } else {
                const sht_status_t ss = sweep(st);
                if (ss != SHT_OK) return ss;
            }
            timing_end(pl, t, st);
        }
        if (gexec) cudaGraphExecDestroy(gexec);          // released once its queued launches have run
    }
    return SHT_OK;
}

// second workspace of the T_m-space iterations (folded T_m of the input maps) + uncovered-power table; the padded map
// columns must stay finite, so the workspace is zero-filled once, on stream `st` (ordered before the caller's kernels)
static void iter_reserve(sht_plan_t pl, cudaStream_t st)
{
    const DevicePlan& d = pl->d;
    const size_t ubytes = (size_t)d.nh * d.ncomp * d.kpad * sizeof(double);
    double *fm = nullptr, *up = nullptr;
    if (cudaMalloc((void**)&fm, pl->F_bytes) != cudaSuccess || cudaMalloc((void**)&up, ubytes) != cudaSuccess ||
        cudaMemsetAsync(fm, 0, pl->F_bytes, st) != cudaSuccess) {
        cudaGetLastError();
        if (fm) cudaFree(fm);
        if (up) cudaFree(up);
        pl->iter_reserve_failed = true;                  // do not retry on every call: fall back to residual maps
        return;
    }
    pl->Fmap = fm; pl->upow = up;
}

extern "C" sht_status_t sht_analysis_iter(sht_plan_t pl, const double* maps, double* alm, int niter,
                                          double* resid_rms, void* stream)
{
    NvtxRange nvtx_entry("sht_analysis_iter");
    if (!pl) return SHT_ERR_NULL;
    if (!maps || !alm) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    if (niter < 0) { snprintf(pl->err, sizeof(pl->err), "niter < 0"); return SHT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const DevicePlan& d = pl->d;
    if (niter > 0 && pl->iter_mode != SHT_ITER_PIXEL) {
        // second workspace: normally reserved ahead (sht_plan_reserve_iter); otherwise allocated here, which is the one
        // place a device entry may synchronise (cudaMalloc) -- its zero fill is ordered on the caller's stream
        if (!pl->Fmap && !pl->iter_reserve_failed) iter_reserve(pl, st);
        if (pl->iter_mode == SHT_ITER_IMMEDIATE) {
            if (!pl->Fmap) { snprintf(pl->err, sizeof(pl->err), "immediate iteration: no memory for the second workspace"); return SHT_ERR_CUDA; }
            return iter_immediate(pl, maps, alm, niter, resid_rms, st);
        }
        if (pl->Fmap) return iter_tm_space(pl, maps, alm, niter, resid_rms, st);
    }
    // residual maps of one chunk + sum-of-squares accumulators (stream-ordered scratch)
    AsyncScratch ress(st), accs(st);
    if (niter > 0) {
        SHT_TRY(ress.alloc((size_t)pl->chunk * d.ncomp * d.npix * sizeof(double)), "residual scratch");
        SHT_TRY(accs.alloc((size_t)pl->chunk * d.ncomp * sizeof(double)), "rms scratch");
    }
    double* res = ress.d(); double* acc = accs.d();
    sht_status_t s = SHT_OK;
    for (int k0 = 0; k0 < pl->nmaps && s == SHT_OK; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        s = analysis_chunk(pl, pl->d, maps, k0, alm, k0, pl->F, kmaps, false, st);
        for (int it = 0; it < niter && s == SHT_OK; ++it) {
            // r = map - synthesis(a): `res` is indexed from the chunk start, maps/alm from map 0
            s = synthesis_chunk(pl, pl->d, alm, k0, res, 0, pl->F, kmaps, maps, k0, st);
            if (s != SHT_OK) break;
            if (resid_rms) {
                const int nrow = kmaps * d.ncomp;
                SHT_TRY(cudaMemsetAsync(acc, 0, (size_t)nrow * sizeof(double), st), "rms memset");
                dim3 grid(64, nrow < 65535 ? nrow : 65535);
                k_sumsq<<<grid, 256, 0, st>>>(res, d.npix, nrow, acc);
                k_rms_finish<<<(nrow + 127) / 128, 128, 0, st>>>(acc, nrow, 1.0 / (double)d.npix,
                                                                 resid_rms + (size_t)it * pl->nmaps * d.ncomp + (size_t)k0 * d.ncomp);
                pl->launches += 2;
                SHT_TRY(cudaGetLastError(), "rms kernels");
            }
            s = analysis_chunk(pl, pl->d, res, 0, alm, k0, pl->F, kmaps, true, st);
        }
    }
    return s;
}

extern "C" sht_status_t sht_plan_reserve_iter(sht_plan_t pl)
{
    if (!pl) return SHT_ERR_NULL;
    if (pl->Fmap) return SHT_OK;
    pl->iter_reserve_failed = false;
    iter_reserve(pl, nullptr);
    if (!pl->Fmap) { snprintf(pl->err, sizeof(pl->err), "no memory for the second workspace"); return SHT_ERR_ALLOC; }
    if (cudaStreamSynchronize(nullptr) != cudaSuccess) return cuda_fail(pl, "reserve sync", cudaGetLastError());
    return SHT_OK;
}

// Pixel-domain E/B decomposition (eq. 16 / 19): S^{E,B} = (F^t lambda^{E,B} F) S.  Per chunk: ring FFTs
// of (Q,U) -> single-component Legendre analysis (item 9: half of the block products) -> the a_lm of that component stay
// in a stream-ordered scratch -> single-component Legendre synthesis -> backward ring FFTs.
extern "C" sht_status_t sht_eb_split(sht_plan_t pl, const double* maps_in, double* maps_out, int which, void* stream)
{
    if (!pl) return SHT_ERR_NULL;
    if (!maps_in || !maps_out) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    if (pl->d.spin != 2 || (which != SHT_POL_E && which != SHT_POL_B)) {
        snprintf(pl->err, sizeof(pl->err), "sht_eb_split needs a spin-2 plan and which = SHT_POL_E or SHT_POL_B");
        return SHT_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    AsyncScratch as(st);
    SHT_TRY(as.alloc((size_t)pl->chunk * pl->d.nalm * 2 * sizeof(double)), "a_lm scratch");
    sht_status_t s = SHT_OK;
    for (int k0 = 0; k0 < pl->nmaps && s == SHT_OK; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        s = analysis_chunk(pl, pl->d, maps_in, k0, as.d(), 0, pl->F, kmaps, false, st, which);
        if (s == SHT_OK) s = synthesis_chunk(pl, pl->d, as.d(), 0, maps_out, k0, pl->F, kmaps, nullptr, 0, st, which);
    }
    return s;
}

extern "C" sht_status_t sht_plan_set_iter_mode(sht_plan_t pl, int mode)
{
    if (!pl) return SHT_ERR_NULL;
    if (mode != SHT_ITER_TM && mode != SHT_ITER_PIXEL && mode != SHT_ITER_IMMEDIATE) return SHT_ERR_INVALID_ARG;
    pl->iter_mode = mode;
    return SHT_OK;
}

// ---- host-buffer entries: chunked H2D -> transform -> D2H, up to four chunks in flight -----------------
// Each chunk has its own stream, staging buffers and slice of the workspace, so the upload of chunk i+2 does not
// wait for the download of chunk i (PCIe is full duplex; with two slots the uploads queued behind the downloads).
static sht_status_t host_setup(sht_plan_t pl)
{
    if (pl->host_ready) return SHT_OK;
    const DevicePlan& d = pl->d;
    // chunk size: about a sixteenth of the maps (the first upload and the last download of a call are not overlapped:
    // short chunks keep that fill and drain small; 882 -> 968 maps/s end to end at config 3 against chunks of an eighth),
    // a multiple of the k-tile, and small enough for host_nb workspace slices
    int nb = d.kpad / KTILE_MAPS;
    if (nb > 4) nb = 4;
    if (nb < 1) nb = 1;
    int hc;
    if (nb > 1) {
        hc = ((pl->nmaps / 16 + KTILE_MAPS - 1) / KTILE_MAPS) * KTILE_MAPS;
        if (hc < KTILE_MAPS) hc = KTILE_MAPS;
        const int cap = d.kpad / nb / KTILE_MAPS * KTILE_MAPS;
        if (hc > cap) hc = cap;
        pl->host_kpad = hc;
    } else {
        hc = pl->chunk;
        pl->host_kpad = d.kpad;
    }
    pl->host_chunk = hc;
    pl->host_nb = nb;
    const size_t mbytes = (size_t)hc * d.ncomp * d.npix * sizeof(double);
    const size_t abytes = (size_t)hc * d.ncomp * d.nalm * 2 * sizeof(double);
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < nb && e == cudaSuccess; ++i) {
        e = cudaMalloc((void**)&pl->stage_maps[i], mbytes);
        if (e == cudaSuccess) e = cudaMalloc((void**)&pl->stage_alm[i], abytes);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&pl->hstream[i], cudaStreamNonBlocking);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pl->hevent, cudaEventDisableTiming);
    if (e != cudaSuccess) {                              // nothing half-built stays behind: the next call starts over
        for (int i = 0; i < 4; ++i) {
            if (pl->stage_maps[i]) { cudaFree(pl->stage_maps[i]); pl->stage_maps[i] = nullptr; }
            if (pl->stage_alm[i]) { cudaFree(pl->stage_alm[i]); pl->stage_alm[i] = nullptr; }
            if (pl->hstream[i]) { cudaStreamDestroy(pl->hstream[i]); pl->hstream[i] = nullptr; }
        }
        if (pl->hevent) { cudaEventDestroy(pl->hevent); pl->hevent = nullptr; }
        return cuda_fail(pl, "host-path staging", e);
    }
    pl->host_ready = true;
    return SHT_OK;
}

static sht_status_t host_run(sht_plan_t pl, const double* in_host, double* out_host, bool analysis)
{
    NvtxRange nvtx_entry("sht host entry (chunked H2D / transform / D2H)");
    if (!pl) return SHT_ERR_NULL;
    if (!in_host || !out_host) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    sht_status_t s = host_setup(pl);
    if (s != SHT_OK) return s;
    const DevicePlan& d = pl->d;
    const size_t map_elems = (size_t)d.ncomp * d.npix, alm_elems = (size_t)d.ncomp * d.nalm * 2;
    const size_t in_elems = analysis ? map_elems : alm_elems, out_elems = analysis ? alm_elems : map_elems;
    DevicePlan dh = d;
    dh.kpad = pl->host_kpad;
    dh.nkg = dh.kpad / KG;
    const size_t f_slice = (size_t)d.nh * (d.lmax + 1) * d.ncomp * 2 * pl->host_kpad * 2;   // doubles per chunk workspace
    // the chunk streams share the plan's workspace and lambda scratch with the device entries: wait for whatever the
    // caller queued before (the host entries are synchronous calls anyway)
    SHT_TRY(cudaDeviceSynchronize(), "host-path entry sync");
    // staged mode: the lambda blocks of this direction are generated once, on the first chunk stream; the other
    // streams wait for them and every chunk launches the contraction kernel only
    SHT_TRY(launch_lambda_blocks(pl, dh, analysis, pl->hstream[0]), "lambda blocks");
    SHT_TRY(cudaEventRecord(pl->hevent, pl->hstream[0]), "lambda event");
    for (int i = 1; i < pl->host_nb; ++i) SHT_TRY(cudaStreamWaitEvent(pl->hstream[i], pl->hevent, 0), "lambda wait");
    int idx = 0;
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->host_chunk, ++idx) {
        const int b = idx % pl->host_nb;
        const int kmaps = pl->nmaps - k0 < pl->host_chunk ? pl->nmaps - k0 : pl->host_chunk;
        cudaStream_t st = pl->hstream[b];
        double* dmaps = pl->stage_maps[b]; double* dalm = pl->stage_alm[b];
        double* din = analysis ? dmaps : dalm; double* dout = analysis ? dalm : dmaps;
        double* F = pl->F + (size_t)b * f_slice;
        SHT_TRY(cudaMemcpyAsync(din, in_host + (size_t)k0 * in_elems, (size_t)kmaps * in_elems * sizeof(double),
                                cudaMemcpyHostToDevice, st), "H2D");
        // staging buffers are indexed from the chunk start: pass k0 = 0
        s = analysis ? analysis_chunk(pl, dh, dmaps, 0, dalm, 0, F, kmaps, false, st, 0, false)
                     : synthesis_chunk(pl, dh, dalm, 0, dmaps, 0, F, kmaps, nullptr, 0, st, 0, false);
        if (s != SHT_OK) return s;
        SHT_TRY(cudaMemcpyAsync(out_host + (size_t)k0 * out_elems, dout, (size_t)kmaps * out_elems * sizeof(double),
                                cudaMemcpyDeviceToHost, st), "D2H");
    }
    for (int i = 0; i < pl->host_nb; ++i) SHT_TRY(cudaStreamSynchronize(pl->hstream[i]), "host-path sync");
    return SHT_OK;
}

extern "C" sht_status_t sht_analysis_host(sht_plan_t pl, const double* maps_host, double* alm_host)
{
    return host_run(pl, maps_host, alm_host, true);
}

extern "C" sht_status_t sht_synthesis_host(sht_plan_t pl, const double* alm_host, double* maps_host)
{
    return host_run(pl, alm_host, maps_host, false);
}

// ---- FP32 storage at the ABI (include/sht.h): widen -> FP64 transform -> round, chunk by chunk -----------------
// pairs of values per thread (every row length here is even: npix = 12 nside^2, a_lm rows are (re, im) pairs)
__global__ void __launch_bounds__(256) k_widen_f32(const float2* __restrict__ in, double2* __restrict__ out, size_t npair)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npair; i += (size_t)gridDim.x * blockDim.x) {
        const float2 v = in[i];
        out[i] = make_double2((double)v.x, (double)v.y);
    }
}
__global__ void __launch_bounds__(256) k_round_f32(const double2* __restrict__ in, float2* __restrict__ out, size_t npair)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npair; i += (size_t)gridDim.x * blockDim.x) {
        const double2 v = in[i];
        out[i] = make_float2((float)v.x, (float)v.y);            // round to nearest even
    }
}
static unsigned f32_grid(size_t npair) { const size_t g = (npair + 255) / 256; return (unsigned)(g < 8192 ? (g ? g : 1) : 8192); }

// single-precision staging of the host entries (one pair of buffers per chunk slot), allocated on the first such call
static sht_status_t host_setup_f32(sht_plan_t pl)
{
    if (pl->host_f32_ready) return SHT_OK;
    const DevicePlan& d = pl->d;
    const size_t mbytes = (size_t)pl->host_chunk * d.ncomp * d.npix * sizeof(float);
    const size_t abytes = (size_t)pl->host_chunk * d.ncomp * d.nalm * 2 * sizeof(float);
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < pl->host_nb && e == cudaSuccess; ++i) {
        e = cudaMalloc((void**)&pl->stage_maps_f32[i], mbytes);
        if (e == cudaSuccess) e = cudaMalloc((void**)&pl->stage_alm_f32[i], abytes);
    }
    if (e != cudaSuccess) {
        for (int i = 0; i < 4; ++i) {
            if (pl->stage_maps_f32[i]) { cudaFree(pl->stage_maps_f32[i]); pl->stage_maps_f32[i] = nullptr; }
            if (pl->stage_alm_f32[i]) { cudaFree(pl->stage_alm_f32[i]); pl->stage_alm_f32[i] = nullptr; }
        }
        return cuda_fail(pl, "single-precision staging", e);
    }
    pl->host_f32_ready = true;
    return SHT_OK;
}

// host = true: `in` / `out` are host pointers, chunks pipelined over the plan's streams as in host_run; host = false: device
// pointers, every chunk on the caller's stream through staging slot 0
static sht_status_t run_f32(sht_plan_t pl, const float* in, float* out, bool analysis, bool host, cudaStream_t user_st)
{
    if (!pl) return SHT_ERR_NULL;
    if (!in || !out) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    sht_status_t s = host_setup(pl);
    if (s == SHT_OK && host) s = host_setup_f32(pl);
    if (s != SHT_OK) return s;
    const DevicePlan& d = pl->d;
    const size_t map_elems = (size_t)d.ncomp * d.npix, alm_elems = (size_t)d.ncomp * d.nalm * 2;
    const size_t in_elems = analysis ? map_elems : alm_elems, out_elems = analysis ? alm_elems : map_elems;
    DevicePlan dh = d;
    dh.kpad = pl->host_kpad;
    dh.nkg = dh.kpad / KG;
    const size_t f_slice = (size_t)d.nh * (d.lmax + 1) * d.ncomp * 2 * pl->host_kpad * 2;
    if (host) {
        SHT_TRY(cudaDeviceSynchronize(), "host-path entry sync");
        SHT_TRY(launch_lambda_blocks(pl, dh, analysis, pl->hstream[0]), "lambda blocks");
        SHT_TRY(cudaEventRecord(pl->hevent, pl->hstream[0]), "lambda event");
        for (int i = 1; i < pl->host_nb; ++i) SHT_TRY(cudaStreamWaitEvent(pl->hstream[i], pl->hevent, 0), "lambda wait");
    } else {
        SHT_TRY(launch_lambda_blocks(pl, dh, analysis, user_st), "lambda blocks");
    }
    int idx = 0;
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->host_chunk, ++idx) {
        const int b = host ? idx % pl->host_nb : 0;
        const int kmaps = pl->nmaps - k0 < pl->host_chunk ? pl->nmaps - k0 : pl->host_chunk;
        cudaStream_t st = host ? pl->hstream[b] : user_st;
        double* dmaps = pl->stage_maps[b]; double* dalm = pl->stage_alm[b];
        double* din = analysis ? dmaps : dalm; double* dout = analysis ? dalm : dmaps;
        double* F = pl->F + (size_t)b * f_slice;
        const size_t nin = (size_t)kmaps * in_elems, nout = (size_t)kmaps * out_elems;
        const float* src = in + (size_t)k0 * in_elems;
        float* dst = out + (size_t)k0 * out_elems;
        if (host) {
            float* fin = analysis ? pl->stage_maps_f32[b] : pl->stage_alm_f32[b];
            SHT_TRY(cudaMemcpyAsync(fin, src, nin * sizeof(float), cudaMemcpyHostToDevice, st), "H2D");
            src = fin;
        }
        k_widen_f32<<<f32_grid(nin / 2), 256, 0, st>>>(reinterpret_cast<const float2*>(src), reinterpret_cast<double2*>(din), nin / 2);
        pl->launches++;
        SHT_TRY(cudaGetLastError(), "widen kernel");
        s = analysis ? analysis_chunk(pl, dh, dmaps, 0, dalm, 0, F, kmaps, false, st, 0, false)
                     : synthesis_chunk(pl, dh, dalm, 0, dmaps, 0, F, kmaps, nullptr, 0, st, 0, false);
        if (s != SHT_OK) return s;
        float* fout = host ? (analysis ? pl->stage_alm_f32[b] : pl->stage_maps_f32[b]) : dst;
        k_round_f32<<<f32_grid(nout / 2), 256, 0, st>>>(reinterpret_cast<const double2*>(dout), reinterpret_cast<float2*>(fout), nout / 2);
        pl->launches++;
        SHT_TRY(cudaGetLastError(), "round kernel");
        if (host) SHT_TRY(cudaMemcpyAsync(dst, fout, nout * sizeof(float), cudaMemcpyDeviceToHost, st), "D2H");
    }
    if (host)
        for (int i = 0; i < pl->host_nb; ++i) SHT_TRY(cudaStreamSynchronize(pl->hstream[i]), "host-path sync");
    return SHT_OK;
}

extern "C" sht_status_t sht_analysis_f32(sht_plan_t pl, const float* maps, float* alm, void* stream)
{
    return run_f32(pl, maps, alm, true, false, (cudaStream_t)stream);
}
extern "C" sht_status_t sht_synthesis_f32(sht_plan_t pl, const float* alm, float* maps, void* stream)
{
    return run_f32(pl, alm, maps, false, false, (cudaStream_t)stream);
}
extern "C" sht_status_t sht_analysis_host_f32(sht_plan_t pl, const float* maps_host, float* alm_host)
{
    return run_f32(pl, maps_host, alm_host, true, true, nullptr);
}
extern "C" sht_status_t sht_synthesis_host_f32(sht_plan_t pl, const float* alm_host, float* maps_host)
{
    return run_f32(pl, alm_host, maps_host, false, true, nullptr);
}

// ---- eq. A7 packed real-square a_lm format -----------------------------------------------------------------
static sht_status_t a7_run(int lmax, long long rows, double* alm, double* sq, bool pack, void* stream)
{
    if (!alm || !sq) return SHT_ERR_NULL;
    if (lmax < 0 || lmax > 16383 || rows < 0) return SHT_ERR_INVALID_ARG;
    if (rows == 0) return SHT_OK;
    const long long nalm = (long long)(lmax + 1) * (lmax + 2) / 2, total = rows * nalm;
    const unsigned grid = (unsigned)((total + 255) / 256);
    if (pack) k_a7<true><<<grid, 256, 0, (cudaStream_t)stream>>>(lmax, nalm, rows, alm, sq);
    else k_a7<false><<<grid, 256, 0, (cudaStream_t)stream>>>(lmax, nalm, rows, alm, sq);
    return cudaGetLastError() == cudaSuccess ? SHT_OK : SHT_ERR_CUDA;
}

extern "C" sht_status_t sht_alm_pack_a7(int lmax, long long rows, const double* alm, double* packed, void* stream)
{
    return a7_run(lmax, rows, const_cast<double*>(alm), packed, true, stream);
}

extern "C" sht_status_t sht_alm_unpack_a7(int lmax, long long rows, const double* packed, double* alm, void* stream)
{
    return a7_run(lmax, rows, alm, const_cast<double*>(packed), false, stream);
}

extern "C" sht_status_t sht_plan_set_lambda_mode(sht_plan_t pl, int mode)
{
    if (!pl) return SHT_ERR_NULL;
    if (mode != SHT_LAMBDA_FUSED && mode != SHT_LAMBDA_STAGED) return SHT_ERR_INVALID_ARG;
    if (mode == SHT_LAMBDA_STAGED && !pl->lam) {
        snprintf(pl->err, sizeof(pl->err), "staged lambda mode needs a plan whose scratch fits");
        return SHT_ERR_UNSUPPORTED;
    }
    pl->lam_mode = mode;
    return SHT_OK;
}
extern "C" int sht_plan_lambda_mode(sht_plan_t pl) { return pl ? pl->lam_mode : -1; }

extern "C" sht_status_t sht_plan_set_option(sht_plan_t pl, int option, int value)
{
    if (!pl) return SHT_ERR_NULL;
    if (value < 0) return SHT_ERR_INVALID_ARG;
    switch (option) {
        case SHT_OPT_RING_PATH: pl->fast_ring = value != 0; return SHT_OK;
        case SHT_OPT_LEG_TILES_PER_CTA: pl->leg_tsplit = value; return SHT_OK;
        case SHT_OPT_LEG_RING_SPLIT: pl->leg_nsplit = value < 1 ? 1 : value; return SHT_OK;
        case SHT_OPT_ITER_HYBRID: pl->gs_plain = value == 0; return SHT_OK;
        default: return SHT_ERR_INVALID_ARG;                 // SHT_OPT_ITER_ALIAS_FREE_FROM is read-only
    }
}
extern "C" int sht_plan_get_option(sht_plan_t pl, int option)
{
    if (!pl) return -1;
    switch (option) {
        case SHT_OPT_RING_PATH: return pl->fast_ring ? 1 : 0;
        case SHT_OPT_LEG_TILES_PER_CTA: return pl->leg_tsplit;
        case SHT_OPT_LEG_RING_SPLIT: return pl->leg_nsplit;
        case SHT_OPT_ITER_HYBRID: return pl->gs_plain ? 0 : 1;
        case SHT_OPT_ITER_ALIAS_FREE_FROM: return pl->gs_pstar;
        default: return -1;
    }
}

// ---- introspection -----------------------------------------------------------------------------------
extern "C" long long sht_npix(int nside) { return 12LL * nside * nside; }
extern "C" long long sht_nalm(int lmax) { return (long long)(lmax + 1) * (lmax + 2) / 2; }
extern "C" long long sht_alm_index(int lmax, int l, int m)
{
    if (lmax < 0 || m < 0 || l < m || l > lmax) return -1;
    return (long long)m * (2 * lmax + 1 - m) / 2 + l;
}
extern "C" size_t sht_plan_workspace_bytes(sht_plan_t pl) { return pl ? pl->F_bytes + pl->table_bytes + pl->lam_bytes : 0; }
extern "C" double sht_plan_executed_flops(sht_plan_t pl, int direction)
{
    if (!pl || direction < 0 || direction > 1 || pl->exec_flops_tile[direction] < 0.0) return -1.0;
    double tiles = 0.0;                                  // k-tiles of one call over all internal chunks
    for (int k0 = 0; k0 < pl->nmaps; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        tiles += pl->d.spin == 2 ? (kmaps + KTILE_MAPS / 2 - 1) / (KTILE_MAPS / 2) : (kmaps + KTILE_MAPS - 1) / KTILE_MAPS;   // spin 2: 32 pairs per k-tile
    }
    return tiles * pl->exec_flops_tile[direction];
}
extern "C" int sht_plan_chunk_maps(sht_plan_t pl) { return pl ? pl->chunk : 0; }
extern "C" long long sht_plan_kernel_launches(sht_plan_t pl) { return pl ? pl->launches : 0; }
extern "C" const char* sht_status_string(sht_status_t s)
{
    switch (s) {
        case SHT_OK: return "ok";
        case SHT_ERR_INVALID_ARG: return "invalid argument";
        case SHT_ERR_UNSUPPORTED: return "unsupported configuration";
        case SHT_ERR_ALLOC: return "allocation failed";
        case SHT_ERR_CUDA: return "CUDA error";
        case SHT_ERR_NULL: return "null pointer";
    }
    return "unknown status";
}
extern "C" const char* sht_last_error(sht_plan_t pl) { return pl ? pl->err : ""; }

extern "C" double sht_measure_fp64_mma_peak(double ms)
{
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1.0;
    const int threads = 512, iters = 4000;
    double* out = nullptr;
    if (cudaMalloc((void**)&out, (size_t)nsm * threads * sizeof(double)) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_mma_peak<<<nsm, threads>>>(out, iters);                     // warm-up
    cudaDeviceSynchronize();
    const double flops_per_launch = (double)nsm * (threads / 32) * iters * 16.0 * 512.0;
    double best = -1.0, elapsed = 0.0;
    // launches back to back until `ms` of device time has passed; report the sustained rate
    int n = 0;
    cudaEventRecord(e0);
    while (elapsed < ms && n < 100000) {
        for (int r = 0; r < 8; ++r) k_mma_peak<<<nsm, threads>>>(out, iters);
        n += 8;
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        elapsed = t;
    }
    if (elapsed > 0.0 && cudaGetLastError() == cudaSuccess) best = flops_per_launch * n / (elapsed * 1e-3) * 1e-12;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return best;
}

// ---- sht_eb_split without any allocation (include/sht.h) ------------------------------------------------
// The a_lm scratch of one chunk lives in a file-scope device array instead of a stream-ordered allocation.  In host code
// `g_eb_static_scratch` is only a stand-in for the symbol, not a device address: the kernels get the pointer that
// cudaGetSymbolAddress returns for the CURRENT device (every device that loads the module has its own copy), looked up
// once per device and kept in g_eb_static_ptr[].
static __device__ __align__(256) double g_eb_static_scratch[SHT_EB_STATIC_MAX_BYTES / sizeof(double)];
static constexpr int EB_STATIC_MAX_DEVICES = 64;
static double* g_eb_static_ptr[EB_STATIC_MAX_DEVICES];   // per device ordinal; written once (same value from any thread)

static cudaError_t eb_static_scratch(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= EB_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    double* p = __atomic_load_n(&g_eb_static_ptr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, g_eb_static_scratch);
        if (e != cudaSuccess) return e;
        __atomic_store_n(&g_eb_static_ptr[dev], p, __ATOMIC_RELEASE);
    }
    *out = p;
    return cudaSuccess;
}

extern "C" sht_status_t sht_eb_split_static(sht_plan_t pl, const double* maps_in, double* maps_out, int which, void* stream)
{
    if (!pl) return SHT_ERR_NULL;
    if (!maps_in || !maps_out) { snprintf(pl->err, sizeof(pl->err), "null data pointer"); return SHT_ERR_NULL; }
    if (pl->d.spin != 2 || (which != SHT_POL_E && which != SHT_POL_B)) {
        snprintf(pl->err, sizeof(pl->err), "sht_eb_split_static needs a spin-2 plan and which = SHT_POL_E or SHT_POL_B");
        return SHT_ERR_INVALID_ARG;
    }
    const size_t need = (size_t)pl->chunk * pl->d.nalm * 2 * sizeof(double);
    if (need > (size_t)SHT_EB_STATIC_MAX_BYTES) {
        snprintf(pl->err, sizeof(pl->err),
                 "sht_eb_split_static: the a_lm scratch of one chunk (%d maps x %lld a_lm x 16 B = %zu bytes) exceeds the static "
                 "array (SHT_EB_STATIC_MAX_BYTES = %zu bytes); use fewer maps per plan or sht_eb_split",
                 pl->chunk, (long long)pl->d.nalm, need, (size_t)SHT_EB_STATIC_MAX_BYTES);
        return SHT_ERR_INVALID_ARG;
    }
    double* scratch = nullptr;
    SHT_TRY(eb_static_scratch(&scratch), "address of the static a_lm scratch");
    cudaStream_t st = (cudaStream_t)stream;
    sht_status_t s = SHT_OK;
    for (int k0 = 0; k0 < pl->nmaps && s == SHT_OK; k0 += pl->chunk) {
        const int kmaps = pl->nmaps - k0 < pl->chunk ? pl->nmaps - k0 : pl->chunk;
        s = analysis_chunk(pl, pl->d, maps_in, k0, scratch, 0, pl->F, kmaps, false, st, which);
        if (s == SHT_OK) s = synthesis_chunk(pl, pl->d, scratch, 0, maps_out, k0, pl->F, kmaps, nullptr, 0, st, which);
    }
    return s;
}
