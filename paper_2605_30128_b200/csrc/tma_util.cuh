// TMA / mbarrier helpers, launch-argument structs and tensor-map builders shared by the cell kernels
// (cell_march.cu: FP32-product march kernel; cell_xyz.cu: the line-owned x/y/z kernel).
#pragma once
#include <cuda.h>

#include "chfsi_internal.h"

namespace chfsi {

struct MarchArgs {
    int nc[3], n1[3];
    int has_phase;
    int phd[3];                 // direction d has a nontrivial Bloch phase (phi_d != 1)
    double ph_re[3], ph_im[3];
    int nseg, cps;              // z segments, cells per segment
    int nvec, nchunks;
    int useR;
    const double* fields;       // [M][4] = V+Bz, V-Bz, Bx, By
    const double* cin;          // [nvec]
    const double* cR;           // [nvec] or null
    double* out;
    long long ld_out;
};

// Tensor maps of one launch.  main/face[0]: n lines, [1]: P lines, [2]: 1 line (the y-wrapped line of the last cell row).
// (cell_mma.cu uses the same struct with its own boxes: main[0..2] = (C/2, 2(P+1) rows, P+1 / P / 1 lines), face[0] =
// (C/2, 2P rows, 1 line), face[1] = (C/2, 2 rows, 1 line).)
struct MarchMaps {
    CUtensorMap main[3];    // box (C/2 doubles, 2P rows, lines) of `in`
    CUtensorMap face[3];    // box (C/2 doubles, 2 rows, lines) of `in`: the x = P column
    CUtensorMap R;          // box (C/2 doubles, 2P rows, P lines) of R
    CUtensorMap F;          // box (4P doubles, P lines) of the packed fields
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    uint32_t ok = 0;
    const uint32_t a = smem_u32(b);
    while (!ok) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
// the same with an L2 eviction-priority hint: the packed node fields are re-read by every vector chunk, so they are
// loaded evict_last and stay in L2 while the multivectors stream through
__device__ __forceinline__ void tma_load_2d_hint(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(policy) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static inline EncodeFn get_encode() {
    static EncodeFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeFn>(p);
    }
    return fn;
}

// 3-D view of a multivector: dim0 = the 2*nvec reals of one (node, spin) row that belong to this launch (the row pitch
// is ld complex elements; columns at and beyond nvec are out of bounds for TMA and arrive as zeros, so a box never reads
// past the caller's allocation whatever ld and the chunk offset are), dim1 = the 2*N1x rows of one x-line, dim2 = the
// N1y*N1z x-lines; box = box_cols reals x box_rows rows x box_lines lines.  f32: the multivector is complex64.
static inline bool make_map3(CUtensorMap* map, const chfsi_mesh* m, const void* base, long long ld, int nvec, int box_cols,
                             int box_rows, int box_lines, bool f32 = false, int swizzle_bytes = 0) {
    EncodeFn enc = get_encode();
    if (!enc) return false;
    const cuuint64_t n1x = (cuuint64_t)m->mc.n1[0];
    const cuuint64_t esz = f32 ? 8 : 16;                        // bytes per complex element
    cuuint64_t gdim[3] = {(cuuint64_t)(2 * (long long)nvec), 2 * n1x, (cuuint64_t)m->mc.n1[1] * (cuuint64_t)m->mc.n1[2]};
    cuuint64_t gstr[2] = {(cuuint64_t)ld * esz, 2 * n1x * (cuuint64_t)ld * esz};
    cuuint32_t box[3] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows, (cuuint32_t)box_lines};
    cuuint32_t estr[3] = {1u, 1u, 1u};
    return enc(map, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), gdim,
               gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 2-D view of the packed fields [M][4]: dim0 = the 4*N1x doubles of one x-line, dim1 = lines; box = 4P doubles x P lines
// (f32: the FP32 copy of the fields)
static inline bool make_mapF(CUtensorMap* map, const chfsi_mesh* m, int P, bool f32 = false) {
    EncodeFn enc = get_encode();
    if (!enc) return false;
    const cuuint64_t n1x = (cuuint64_t)m->mc.n1[0];
    cuuint64_t gdim[2] = {4 * n1x, (cuuint64_t)m->mc.n1[1] * (cuuint64_t)m->mc.n1[2]};
    cuuint64_t gstr[1] = {n1x * (f32 ? 16u : 32u)};
    cuuint32_t box[2] = {(cuuint32_t)(4 * P), (cuuint32_t)P};
    cuuint32_t estr[2] = {1u, 1u};
    return enc(map, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, f32 ? (void*)m->dF32 : (void*)m->dF, gdim, gstr,
               box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}


}  // namespace chfsi
