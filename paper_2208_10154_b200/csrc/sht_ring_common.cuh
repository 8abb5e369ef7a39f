// sht_ring_common.cuh -- helpers shared by the ring kernels that move their data with bulk copies and TMA
// (sht_ring_pow2.cu, sht_ring_mixed.cu): async-proxy fences, bulk-group waits, 5-D tensor-map loads / stores of the
// workspace lines, and the tensor map itself.
#pragma once
#include "sht_legendre_common.cuh"

namespace sht {
namespace p2 {

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }

__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int NKEEP>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(NKEEP) : "memory"); }
template <int NKEEP>
__device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(NKEEP) : "memory"); }
__device__ __forceinline__ void tma_store_5d(const CUtensorMap* map, const void* src, int c0, int c1, int c2, int c3, int c4)
{
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
                 : "memory");
}
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
        : "memory");
}

}  // namespace p2

// Workspace F as a 5-D tensor for the ring kernels' boxes of [MB orders] x [E, O] x [KT maps]: innermost the 2 KT
// doubles of KT maps (re, im); c = which KT-map part of the 4-map line; ch = 2 comp + h; m; (p, kg).
// planes: dimension order (doubles, m, ch, c, pkg) -> box lands as [h][m][map] (conflict-free staging); otherwise
// ascending strides (doubles, c, ch, m, pkg) -> [m][h][map].
inline cudaError_t make_tmap_ring(const DevicePlan& d, const double* F, int kt, int mb, bool planes, CUtensorMap* tm)
{
    PFN_tmapEncodeTiled enc = tmap_encoder();
    if (!enc) return cudaErrorNotSupported;
    const cuuint64_t line = 128, mstr = (cuuint64_t)d.ncomp * line, pstr = (cuuint64_t)(d.lmax + 1) * mstr;
    const cuuint64_t n_m = (cuuint64_t)d.lmax + 1, n_ch = 2 * (cuuint64_t)d.ncomp, n_c = (cuuint64_t)(KG / kt),
                     n_pkg = (cuuint64_t)d.nh * d.nkg;
    cuuint64_t dims[5], strides[4];
    cuuint32_t box[5];
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    dims[0] = 2 * (cuuint64_t)kt; box[0] = 2 * (cuuint32_t)kt;
    if (planes) {
        dims[1] = n_m; strides[0] = mstr; box[1] = (cuuint32_t)mb;
        dims[2] = n_ch; strides[1] = 64; box[2] = 2;
        dims[3] = n_c; strides[2] = (cuuint64_t)kt * 16; box[3] = 1;
    } else {
        dims[1] = n_c; strides[0] = (cuuint64_t)kt * 16; box[1] = 1;
        dims[2] = n_ch; strides[1] = 64; box[2] = 2;
        dims[3] = n_m; strides[2] = mstr; box[3] = (cuuint32_t)mb;
    }
    dims[4] = n_pkg; strides[3] = pstr; box[4] = 1;
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<double*>(F), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

}  // namespace sht
