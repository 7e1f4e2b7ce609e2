// wl_small.cu -- the SMALL multigrid levels (at most 4096 cells per block of the launch) entirely on chip.
//
// Below the bandwidth-relevant levels a V-cycle (readings R-S, R-T, R-T2 of DESIGN.md) is a chain
// of short dependent passes: restrict, six Jacobi-PCG iterations with two dot products each, prolong -- per level.
// Run through global memory, every pass costs a few dependent L2 round trips plus a grid-wide barrier (3-4 us);
// the paper calls these reductions "rather inefficient".  k_small runs the whole chain of a group of small
// levels as ONE launch of ONE thread-block cluster (1, 2, 4, 8 or 16 blocks of 1024 threads):
//   * a block owns a contiguous chunk of 4096 cells of the level, four cells per thread; x, r, q = A e and 1/D of a
//     cell live in its thread's registers for the whole smoother call, the face coefficients and the CG direction e in
//     the block's shared memory;
//   * the stencil reads e of cells owned by another block through distributed shared memory;
//   * a dot product is a block reduction (shuffles + shared memory) followed, in a multi-block cluster, by one hardware
//     cluster barrier and a fixed-order sum of the blocks' partials read through distributed shared memory: every block
//     obtains the same bits and takes the same branches of the R-T guards;
//   * restriction and prolongation between two levels go through the level arrays in global memory (L2), one pass and
//     one cluster barrier each.
// Nothing here depends on the order in which blocks are scheduled; sums are taken in a fixed order (bit-reproducible).
#include <cstdio>
#include "wl_internal.h"
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

#define SM_NT 1024                     // threads per block
#define SM_K 4                         // cells per thread, at most
#define SM_CHUNK (SM_NT * SM_K)        // cells per block, at most
#define SM_ONE 2048                    // a level of at most this many cells is smoothed by ONE block (block barriers only)

struct SmShared {
    float e[SM_CHUNK];                 // CG direction of the block's cells (read by the other blocks of the cluster)
    float Llo[3][SM_CHUNK];            // coefficient of the lower / upper face of every cell, per direction
    float Lhi[3][SM_CHUNK];
    unsigned short nlo[3][SM_CHUNK];   // cell numbers (< 65536: at most 16 blocks) of the lower / upper neighbour per direction;
    unsigned short nhi[3][SM_CHUNK];   // across a wall the cell itself (the coefficient is zero there)
    double slots[2][4][16];            // the blocks' partial sums [value][rank], alternating between consecutive reductions
    double warp[4][32];
};

struct SmCtx {
    SmShared* sh;
    int C;                             // blocks in the cluster
    int rank;
    int phase;
    int nt;                            // C == 1: the first nt threads of the block (whole warps) take part in barriers and sums
};

// How a level of N cells is spread over a cluster of C blocks: Cl blocks own 2^shift cells each (1024, 2048 or 4096: one, two or
// four per thread).  A sum over the cluster costs ~1900 cycles, over one block ~900, a stencil sweep ~1100 per cell of a thread:
// up to SM_ONE cells one block does it all; above, as many blocks as give every thread one cell.
__host__ __device__ inline void sm_spread(int N, int C, int& Cl, int& shift)
{
    Cl = 1;
    if (N > SM_ONE) while (Cl * 1024 < N && Cl < C) Cl <<= 1;
    shift = 10;
    while ((Cl << shift) < N && shift < 12) ++shift;
}

__device__ __forceinline__ void sm_bar(int nt)
{
    if (nt >= SM_NT) __syncthreads();
    else if (nt > 32) asm volatile("bar.sync 1, %0;" ::"r"(nt) : "memory");
    else __syncwarp();
}

__device__ __forceinline__ void sm_sync(const SmCtx& c)
{
    if (c.C == 1) sm_bar(c.nt);
    else cg::this_cluster().sync();    // barrier.cluster arrive.release / wait.acquire: orders shared AND global memory in the cluster
}

// sum of NV values over every thread of the cluster; identical bits in every thread.  Contains a cluster-wide barrier.
// Block stage: warp shuffles, one shared-memory hand-over, warp 0 reduces the 32 warp sums.  Cluster stage: warp 0 PUSHES the
// block's sum into slot [rank] of every block's shared memory (remote stores are fire-and-forget; a remote LOAD costs ~350
// cycles and 16 blocks reading 16 slots each queue up behind one another: 4400 against 1900 cycles per reduction, measured),
// one hardware cluster barrier, then every warp adds the C slots of its OWN shared memory in the same fixed tree.
template <int NV>
__device__ __forceinline__ void sm_reduce(SmCtx& c, double (&v)[NV])
{
    SmShared& sh = *c.sh;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double w = warp_red<OpSum>(v[k]);
        if (lane == 0) sh.warp[k][wid] = w;
    }
    if (c.C == 1) {
        const int nw = c.nt >> 5;
        sm_bar(c.nt);
#pragma unroll
        for (int k = 0; k < NV; ++k) v[k] = warp_red<OpSum>(lane < nw ? sh.warp[k][lane] : 0.0);   // one value per lane; every warp redundantly
        sm_bar(c.nt);                                                           // warp[] may be rewritten by the next reduction
        return;
    }
    __syncthreads();
    cg::cluster_group cl = cg::this_cluster();
    double (*slots)[16] = sh.slots[c.phase & 1];
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            const double w = warp_red<OpSum>(sh.warp[k][lane]);
            if (lane < c.C) *cl.map_shared_rank(&slots[k][c.rank], lane) = w;    // lane r -> block r
        }
    }
    cl.sync();                                                                   // every block's sum is in every block's slots
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = warp_red<OpSum>(lane < c.C ? slots[k][lane] : 0.0);     // fixed tree over the ranks
    c.phase++;
}

// cell k of a level (x fastest) -> 0-based coordinates
__device__ __forceinline__ void sm_coords(const Grid& g, int k, int& c0, int& c1, int& c2)
{
    c0 = k % g.n[0];
    const int t = k / g.n[0];
    c1 = t % g.n[1];
    c2 = t / g.n[1];
}
template <int ND>
__device__ __forceinline__ int64_t sm_gidx(const Grid& g, int c0, int c1, int c2)      // 0-based interior coordinates
{
    return (int64_t)WL_OFF + (c0 + 1) + (int64_t)(c1 + 1) * g.sy + (ND == 3 ? (int64_t)(c2 + 1) * g.sz : 0);
}

// prolongation + increment at ONE fine cell (R-S): e = P x_c (piecewise constant) at the cell and its 2 ND neighbours; returns e at the
// cell and, in `acc`, (A_f e) there.  Used by the stand-alone pass (sm_prolong) and by the smoother that absorbs the pass into its
// loading phase: the same expression, so the same bits either way.
template <int ND>
__device__ __forceinline__ float sm_prolong_cell(const LevDev& lf, const LevDev& lc, const int (&cc)[3], int64_t i, float& acc)
{
    const Grid &gf = lf.g, &gc = lc.g;
    const int64_t gst[3] = { 1, gf.sy, gf.sz };
    const float ec = lc.x[sm_gidx<ND>(gc, cc[0] >> 1, cc[1] >> 1, cc[2] >> 1)];
    acc = 0.0f;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        int a[3] = { cc[0], cc[1], cc[2] }, b[3] = { cc[0], cc[1], cc[2] };
        a[d] = cc[d] > 0 ? cc[d] - 1 : (gf.per[d] ? gf.n[d] - 1 : cc[d]);              // across a wall the coefficient is zero
        b[d] = cc[d] < gf.n[d] - 1 ? cc[d] + 1 : (gf.per[d] ? 0 : cc[d]);
        const float el = lc.x[sm_gidx<ND>(gc, a[0] >> 1, a[1] >> 1, a[2] >> 1)];
        const float eh = lc.x[sm_gidx<ND>(gc, b[0] >> 1, b[1] >> 1, b[2] >> 1)];
        acc += lf.L[d * gf.nalloc + i + gst[d]] * (eh - ec) - lf.L[d * gf.nalloc + i] * (ec - el);
    }
    return ec;
}

// ---------------------------------------------------------------- Jacobi-PCG smoother (R-T, R-T2), on chip
//   r <- r - mean(r over the coupled cells) on those cells; z = e = iD r; rho0 = rho = r.z; |rho| < tau: return
//   k = 1..iters: q = A e; gamma = q.e; gamma = 0 or not finite: return; alpha = rho/gamma; x += alpha e; r -= alpha q;
//                 k == iters: return; z = iD r; rho' = r.z; |rho'| < tau or < theta |rho0|: return;
//                 beta = rho'/rho; e = beta e + z; rho = rho'
// Cell k of the block's chunk belongs to thread k mod 1024 (conflict-free shared-memory accesses); the six neighbours of a
// cell are looked up by cell number (tables in shared memory) and read from this block's shared memory or, for the few owned
// by another block, through the cluster window.
template <int ND>
__device__ __forceinline__ void sm_smooth(SmCtx& cl, const LevDev& lv, PcgScal* sc, int iters, const LevDev* coarse)
{
    // coarse != null: the prolongation from that level (x += P x_c, r -= A P x_c) has not been run as a pass of its own and is
    // applied here, while x and r are loaded
    SmShared& sh = *cl.sh;
    const Grid& g = lv.g;
    const int N = g.n[0] * g.n[1] * g.n[2];
    const int tid = threadIdx.x;
    int Cl, shift;
    sm_spread(N, cl.C, Cl, shift);
    const int K = 1 << (shift - 10), cmask = (1 << shift) - 1;        // cells per thread, chunk - 1
    SmCtx c = cl;
    if (Cl == 1) {
        // one block, and of it only the warps that own cells: block-local barriers and sums; everybody else goes straight to the
        // barrier that ends the pass (the caller's)
        c.C = 1;
        c.nt = N >= SM_NT ? SM_NT : (N + 31) & ~31;
        if (cl.rank != 0 || tid >= c.nt) return;
    }
    const int st[3] = { 1, g.n[0], g.n[0] * g.n[1] };
    float x[SM_K], r[SM_K], q[SM_K], d[SM_K];
    bool ok[SM_K];
    auto offset = [&](int k) -> int {          // cell number -> offset into the level arrays (small levels: 32 bits are plenty)
        int c0, c1, c2;
        sm_coords(g, k, c0, c1, c2);
        return (int)sm_gidx<ND>(g, c0, c1, c2);
    };
#pragma unroll
    for (int j = 0; j < SM_K; ++j) {
        const int k = (c.rank << shift) + j * SM_NT + tid, loc = j * SM_NT + tid;
        ok[j] = j < K && k < N;
        x[j] = r[j] = q[j] = d[j] = 0.0f;
        if (!ok[j]) { if (j < K) sh.e[loc] = 0.0f; continue; }
        int cc[3];
        sm_coords(g, k, cc[0], cc[1], cc[2]);
        const int gi = (int)sm_gidx<ND>(g, cc[0], cc[1], cc[2]);
        const int gst[3] = { 1, (int)g.sy, (int)g.sz };
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            // across a wall the neighbour is the cell itself: the coefficient of that face is zero
            sh.nlo[i][loc] = (unsigned short)(cc[i] > 0 ? k - st[i] : (g.per[i] ? k + (g.n[i] - 1) * st[i] : k));
            sh.nhi[i][loc] = (unsigned short)(cc[i] < g.n[i] - 1 ? k + st[i] : (g.per[i] ? k - (g.n[i] - 1) * st[i] : k));
            sh.Llo[i][loc] = lv.L[i * g.nalloc + gi];
            sh.Lhi[i][loc] = lv.L[i * g.nalloc + gi + gst[i]];
        }
        x[j] = lv.x[gi]; r[j] = lv.r[gi]; d[j] = lv.iD[gi];
        if (coarse) {
            float acc;
            const float ec = sm_prolong_cell<ND>(lv, *coarse, cc, gi, acc);
            x[j] += ec;
            r[j] -= acc;
        }
    }
    // operand of the stencil at cell kk: this block's shared memory, or another block's through the cluster window
    auto E = [&](int kk) -> float {
        const int rr = kk >> shift, off = kk & cmask;
        if (rr == c.rank) return sh.e[off];
        return *cg::this_cluster().map_shared_rank(&sh.e[off], rr);
    };
    // ---- R-T2: remove the mean of r over the coupled cells
    double v[2] = { 0.0, 0.0 };
#pragma unroll
    for (int j = 0; j < SM_K; ++j)
        if (ok[j] && d[j] != 0.0f) { v[0] += (double)r[j]; v[1] += 1.0; }
    sm_reduce<2>(c, v);
    const float m = v[1] > 0.0 ? (float)(v[0] / v[1]) : 0.0f;
    double w1[1] = { 0.0 };
#pragma unroll
    for (int j = 0; j < SM_K; ++j) {
        if (d[j] != 0.0f) r[j] -= m;
        const float z = __fmul_rn(d[j], r[j]);
        if (j < K) sh.e[j * SM_NT + tid] = z;
        if (ok[j]) w1[0] += (double)z * (double)r[j];
    }
    sm_reduce<1>(c, w1);                              // (its barrier also publishes e)
    double rho = w1[0];
    const double rho0 = rho;
    int live = 1, done = 0;
    if (fabs(rho) < WL_TAU) live = 0;
    for (int k = 1; k <= iters && live; ++k) {
        double gam[1] = { 0.0 };
#pragma unroll
        for (int j = 0; j < SM_K; ++j) {
            const int loc = j * SM_NT + tid;
            float acc = 0.0f;
            if (ok[j]) {
                const float ec = sh.e[loc];
#pragma unroll
                for (int i = 0; i < ND; ++i) acc += sh.Lhi[i][loc] * (E(sh.nhi[i][loc]) - ec) - sh.Llo[i][loc] * (ec - E(sh.nlo[i][loc]));
                gam[0] += (double)acc * (double)ec;
            }
            q[j] = acc;
        }
        sm_reduce<1>(c, gam);                         // every block has finished reading e
        if (gam[0] == 0.0 || !isfinite(gam[0])) { live = 0; break; }
        const float alpha = (float)(rho / gam[0]);
        double r2[1] = { 0.0 };
#pragma unroll
        for (int j = 0; j < SM_K; ++j) {
            if (j < K) x[j] += alpha * sh.e[j * SM_NT + tid];
            r[j] -= alpha * q[j];
            if (ok[j]) r2[0] += (double)__fmul_rn(d[j], r[j]) * (double)r[j];
        }
        done = k;
        if (k == iters) break;
        sm_reduce<1>(c, r2);
        if (fabs(r2[0]) < WL_TAU || fabs(r2[0]) < WL_THETA * fabs(rho0)) { live = 0; break; }
        const float beta = (float)(r2[0] / rho);
        rho = r2[0];
#pragma unroll
        for (int j = 0; j < SM_K; ++j) {
            const int loc = j * SM_NT + tid;
            if (j < K) sh.e[loc] = __fmaf_rn(beta, sh.e[loc], __fmul_rn(d[j], r[j]));
        }
        sm_sync(c);                                   // the new direction is visible to the whole cluster
    }
#pragma unroll
    for (int j = 0; j < SM_K; ++j)
        if (ok[j]) { const int gi = offset((c.rank << shift) + j * SM_NT + tid); lv.x[gi] = x[j]; lv.r[gi] = r[j]; }
    if (c.rank == 0 && tid == 0) {
        sc->rsum = 0.0; sc->nlive = v[1]; sc->rho = rho; sc->rho0 = rho0; sc->live = live; sc->stop_k = done;
    }
    cl.phase = c.phase;
}

// ---------------------------------------------------------------- residual restriction (R-S): r_c = sum of the 2^n children; x_c = 0
template <int ND>
__device__ __forceinline__ void sm_restrict(const SmCtx& c, const LevDev& lf, const LevDev& lc)
{
    const Grid &gf = lf.g, &gc = lc.g;
    const int N = gc.n[0] * gc.n[1] * gc.n[2];
    for (int k = c.rank * SM_NT + threadIdx.x; k < N; k += c.C * SM_NT) {
        int C0, C1, C2;
        sm_coords(gc, k, C0, C1, C2);
        float s = 0.0f;
#pragma unroll
        for (int a2 = 0; a2 < (ND == 3 ? 2 : 1); ++a2)
#pragma unroll
            for (int a1 = 0; a1 < 2; ++a1) {
                const int64_t b = sm_gidx<ND>(gf, 2 * C0, 2 * C1 + a1, 2 * C2 + a2);
                s += lf.r[b]; s += lf.r[b + 1];
            }
        const int64_t i = sm_gidx<ND>(gc, C0, C1, C2);
        lc.r[i] = s;
        lc.x[i] = 0.0f;
    }
}

// ---------------------------------------------------------------- prolongation + increment (R-S): e = P x_c; x_f += e; r_f -= A_f e
template <int ND>
__device__ __forceinline__ void sm_prolong(const SmCtx& c, const LevDev& lf, const LevDev& lc)
{
    const Grid& gf = lf.g;
    const int N = gf.n[0] * gf.n[1] * gf.n[2];
    for (int k = c.rank * SM_NT + threadIdx.x; k < N; k += c.C * SM_NT) {
        int cc[3];
        sm_coords(gf, k, cc[0], cc[1], cc[2]);
        const int64_t i = sm_gidx<ND>(gf, cc[0], cc[1], cc[2]);
        float acc;
        const float ec = sm_prolong_cell<ND>(lf, lc, cc, i, acc);
        lf.x[i] += ec;
        lf.r[i] -= acc;
    }
}

template <int ND>
__global__ void __launch_bounds__(SM_NT, 1) k_small(const LevDev* levs, const __grid_constant__ CoarseProg prog, DevScal* ds)
{
    extern __shared__ __align__(16) unsigned char sm_raw[];
    __shared__ LevDev la, lb;
    SmCtx c;
    c.sh = reinterpret_cast<SmShared*>(sm_raw);
    c.C = (int)gridDim.x;                               // the launch is one cluster
    c.rank = (int)blockIdx.x;
    c.phase = 0;
    c.nt = SM_NT;
    bool absorbed = false;                              // the previous op was a prolongation left to the smoother that follows it
    for (int o = 0; o < prog.n; ++o) {
        const CoarseOp op = prog.op[o];
        // prolong(l+1 -> l) followed by smooth(l): the smoother loads x and r of level l anyway and applies the prolongation while it
        // does (one pass over the level arrays and one cluster barrier less; the same arithmetic)
        if (op.kind == COP_PROLONG && o + 1 < prog.n && prog.op[o + 1].kind == COP_SMOOTH && prog.op[o + 1].level == op.level) { absorbed = true; continue; }
        if (threadIdx.x == 0) {
            la = levs[op.level];
            lb = levs[op.level + (op.kind == COP_SMOOTH && !absorbed ? 0 : 1)];
        }
        __syncthreads();
        if (op.kind == COP_SMOOTH) { sm_smooth<ND>(c, la, &ds->pcg[op.level], op.iters, absorbed ? &lb : nullptr); absorbed = false; }
        else if (op.kind == COP_RESTRICT) sm_restrict<ND>(c, la, lb);
        else sm_prolong<ND>(c, la, lb);
        sm_sync(c);                                     // the pass's global writes are visible to every block; la / lb are free
    }
}

// ================================================================== host side
// largest cluster (1, 2, 4, 8, 16 blocks) the device can co-schedule for k_small; 0: the kernel cannot run at all
int wl_small_max_cluster(wl_sim* s)
{
    const size_t smem = sizeof(SmShared);
    cudaError_t e;
    if (s->nd == 3) e = cudaFuncSetAttribute(k_small<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    else            e = cudaFuncSetAttribute(k_small<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    if (s->nd == 3) cudaFuncSetAttribute(k_small<3>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    else            cudaFuncSetAttribute(k_small<2>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaGetLastError();
    for (int C = 16; C >= 1; C >>= 1) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(C); cfg.blockDim = dim3(SM_NT); cfg.dynamicSmemBytes = smem; cfg.stream = s->st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n = 0;
        if (s->nd == 3) e = cudaOccupancyMaxActiveClusters(&n, k_small<3>, &cfg);
        else            e = cudaOccupancyMaxActiveClusters(&n, k_small<2>, &cfg);
        if (e == cudaSuccess && n >= 1) return C;
        cudaGetLastError();
    }
    return 0;
}

// blocks of a cluster of at most cmax that k_small spreads a level over (sm_spread); 0: the level is too large for such a cluster
int wl_small_blocks(const Grid& g, int cmax)
{
    const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
    if (cmax < 1 || N > (long long)cmax * SM_CHUNK) return 0;
    int Cl, shift;
    sm_spread((int)N, cmax, Cl, shift);
    return Cl;
}

// one launch: the chain `prog` over small levels, as one cluster of `C` blocks.  Returns 0 if the launch failed.
int wl_k_small_prog(wl_sim* s, const CoarseProg& prog, int C)
{
    if (prog.n <= 0) return 1;
    ProfScope ps_(s, WLK_SMALL, 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C); cfg.blockDim = dim3(SM_NT); cfg.dynamicSmemBytes = sizeof(SmShared); cfg.stream = s->st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    const LevDev* levs = s->levdev;
    DevScal* ds = s->ds;
    cudaError_t e;
    if (s->nd == 3) e = cudaLaunchKernelEx(&cfg, k_small<3>, levs, prog, ds);
    else            e = cudaLaunchKernelEx(&cfg, k_small<2>, levs, prog, ds);
    return e == cudaSuccess;
}
