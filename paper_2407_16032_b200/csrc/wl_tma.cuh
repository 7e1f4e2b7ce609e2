// wl_tma.cuh -- the TMA engine for the stencil kernels of libwl (sm_100a): tensor maps of the padded scalar arrays
// (host), one-instruction box copies into shared memory completing on an mbarrier (device).
#pragma once
#include <cuda.h>
#include <cudaTypedefs.h>
#include "wl_common.cuh"

// ---- bulk asynchronous copies (TMA engine, cp.async.bulk) completing on an mbarrier
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WL_MB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WL_MB_DONE;\n"
        "bra WL_MB_WAIT;\n"
        "WL_MB_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one box of a 3-D tensor map (x fastest) into shared memory; completes `bytes of the box` on the mbarrier
__device__ __forceinline__ void tma_box3(unsigned dst, const CUtensorMap* tm, int c0, int c1, int c2, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}


// Tensor map of one padded scalar array (dims P x S1 x S2 floats, x fastest) with a box of box_x x box_y x 1: one
// tile plane with its halos.  Out-of-range parts of a box are filled with zeros.  Returns 0 when the driver entry
// point is missing or the encoding fails (the caller then takes the cp.async path).
static inline int wl_tensor_map3(CUtensorMap* tm, const float* base, const Grid& g, int box_x, int box_y)
{
    static PFN_cuTensorMapEncodeTiled_v12000 enc = nullptr;
    if (!enc) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn) return 0;
        enc = (PFN_cuTensorMapEncodeTiled_v12000)fn;
    }
    const cuuint64_t dims[3] = { (cuuint64_t)g.P, (cuuint64_t)g.S[1], (cuuint64_t)g.S[2] };
    const cuuint64_t strides[2] = { (cuuint64_t)g.sy * 4, (cuuint64_t)g.sz * 4 };
    const cuuint32_t box[3] = { (cuuint32_t)box_x, (cuuint32_t)box_y, 1 };
    const cuuint32_t es[3] = { 1, 1, 1 };
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-handle cache of encoded tensor maps, keyed by (base pointer, row pitch, box): the solver arrays never move, so every
// map is encoded once (a smoother call used to re-encode ~15 of them) and an encode failure is seen by the caller, which
// then takes the path without TMA.
struct TmCache {
    struct Entry { const float* base; int P, S1, S2, bx, by; CUtensorMap tm; };
    Entry e[64];
    int n;
};
static inline const CUtensorMap* wl_tensor_map_cached(TmCache* c, const float* base, const Grid& g, int box_x, int box_y)
{
    for (int k = 0; k < c->n; ++k) {
        const TmCache::Entry& q = c->e[k];
        if (q.base == base && q.P == g.P && q.S1 == g.S[1] && q.S2 == g.S[2] && q.bx == box_x && q.by == box_y) return &q.tm;
    }
    TmCache::Entry q;
    q.base = base; q.P = g.P; q.S1 = g.S[1]; q.S2 = g.S[2]; q.bx = box_x; q.by = box_y;
    if (!wl_tensor_map3(&q.tm, base, g, box_x, box_y)) return nullptr;
    const int slot = c->n < 64 ? c->n++ : 63;          // a full cache recycles its last slot
    c->e[slot] = q;
    return &c->e[slot].tm;
}

