// wl_vec.cuh -- vector tiles for the whole-grid passes of libwl (sm_100a).
//
// Every fine-grid pass is HBM-bound, so the access pattern is the
// design: one thread owns FOUR consecutive x cells (one 16-byte float4: interior cell c0 = 1
// sits on a 32-byte boundary of its row, wl_common.cuh), a block of 256 threads is LX x LY
// threads (LX = 2^lxl <= 32 along x), and a block marches ZC planes along z keeping the
// z-neighbours of its column in registers.  A tile is therefore (4 LX) x LY x ZC cells; a warp
// reads 512 contiguous bytes per row.  y-neighbours come from L1 (the rows of the adjacent
// threads of the same block), x-neighbours from two scalar loads.
//
// Tiles also carry a mode (TM_GEN / TM_PLB / TM_PLI below): uniform tiles
// (no body within one cell) never load L or iD.
#pragma once
#include "wl_common.cuh"

#define WL_VB 256   // threads per block of every vector-tile kernel

struct VT {
    int lxl;            // log2(threads along x)
    int ngx;            // float4 groups per row = ceil(n0 / 4)
    int ntx, nty, ntz;  // tiles per direction
    int ntiles;
    int zc;             // planes per tile (1 in 2-D)
};

struct VPos {
    int c0, c1;         // first cell of the thread's float4 group; its row
    int z0, z1;         // plane range [z0, z1] of the tile (2-D: 0, 0)
    int nv;             // valid cells in the group (0 = thread idle)
};

__device__ __forceinline__ VPos vt_pos(const Grid& g, const VT& t, int tile)
{
    VPos p;
    const int tid = threadIdx.x;
    const int tx = tid & ((1 << t.lxl) - 1), ty = tid >> t.lxl;
    const int ly = WL_VB >> t.lxl;
    int tix = tile % t.ntx;
    int rem = tile / t.ntx;
    int tiy = rem % t.nty;
    int tiz = rem / t.nty;
    int gx = (tix << t.lxl) + tx;
    p.c0 = 1 + 4 * gx;
    p.c1 = 1 + tiy * ly + ty;
    int nv = g.n[0] - p.c0 + 1;
    nv = nv > 4 ? 4 : nv;
    if (gx >= t.ngx || p.c1 > g.n[1] || nv < 0) nv = 0;
    p.nv = nv;
    if (g.sz == 0) { p.z0 = 0; p.z1 = 0; }
    else {
        p.z0 = 1 + tiz * t.zc;
        p.z1 = p.z0 + t.zc - 1;
        if (p.z1 > g.n[2]) p.z1 = g.n[2];
    }
    return p;
}

// Plain (coherent) loads: the same tile functions run inside the persistent coarse-level kernel,
// where arrays written in an earlier phase by another block are read after a grid barrier; the
// non-coherent path (__ldg) is not allowed there.  In the stand-alone kernels the pointers are
// const __restrict__ kernel parameters and the compiler selects the read-only path itself.
__device__ __forceinline__ float4 ld4(const float* a, int64_t i)
{
    return *reinterpret_cast<const float4*>(a + i);
}
__device__ __forceinline__ float ld1(const float* a, int64_t i) { return a[i]; }

__device__ __forceinline__ void st4(float* __restrict__ a, int64_t i, const float (&v)[4], int nv)
{
    if (nv == 4) *reinterpret_cast<float4*>(a + i) = make_float4(v[0], v[1], v[2], v[3]);
    else
        for (int k = 0; k < nv; ++k) a[i + k] = v[k];
}

__device__ __forceinline__ void unpack4(const float4& v, float (&o)[4]) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }

// row offsets of the y / z neighbours with periodic wrap (solver arrays keep no ghost values)
__device__ __forceinline__ int nb_lo(int c, int n, int per) { return (c == 1 && per) ? n : c - 1; }
__device__ __forceinline__ int nb_hi(int c, int n, int per) { return (c == n && per) ? 1 : c + 1; }

// ---------------------------------------------------------------- tile modes
// Level::plain[tile] (written by k_diag_flags + k_plain_mode after every measure!):
//   TM_GEN  general tile: face coefficients L and the inverse diagonal iD are loaded;
//   TM_PLB  uniform tile (every face coefficient of the tile and of its face-neighbour tiles has its
//           body-free value: Lc inside, 0 on a non-periodic domain boundary, R-O) that touches a
//           non-periodic boundary: L and iD follow from the cell position alone, nothing is loaded;
//   TM_PLI  uniform tile at least one cell away from every non-periodic boundary: L = Lc, iD = iDc.
#define TM_GEN 0
#define TM_PLB 1
#define TM_PLI 2

