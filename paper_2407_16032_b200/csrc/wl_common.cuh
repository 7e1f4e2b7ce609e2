// wl_common.cuh -- shared device-side types of libwl (sm_100a): grid descriptor, index
// helpers, deterministic block/grid reductions, device-resident scalars.
//
// Layout in HBM.  Every field is a padded fp32 array with one ghost
// cell per side (paper layout), x fastest, component-major (SoA).  The x pitch P
// is a multiple of 8 floats and the ghost cell c0 = 0 sits at float offset WL_OFF = 7 of its
// row, so interior cell c0 = 1 starts every row on a 32-byte sector boundary:
//     idx(c0,c1,c2) = WL_OFF + c0 + P*(c1 + S1*c2)
// C index c_d = I_d - 1 of the paper's 1-based padded index I_d; interior c_d = 1..N_d.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define WL_OFF 7
#define WL_MAXLEV 16
#define WL_TAU 1e-30          // PCG guard on |rho|: protects 0/0 only (DESIGN.md R-T)
#define WL_THETA 1e-8         // PCG stops once |rho'| < theta |rho0| (R-T): no CG steps on a converged residual
#define WL_MAX_PARTIALS 2048  // upper bound on the grid size of any reducing kernel

struct Grid {
    int n[3];        // interior cells (n[2] = 1 in 2-D)
    int S[3];        // padded logical sizes n+2 (S[2] = 1 in 2-D)
    int per[3];      // periodic flags
    int P;           // x pitch (floats)
    int64_t sy, sz;  // strides of c1, c2 (sz = 0 in 2-D)
    int64_t nalloc;  // floats per scalar array (multiple of 64)
};

__host__ __device__ __forceinline__ int64_t gidx(const Grid& g, int c0, int c1, int c2)
{
    return (int64_t)WL_OFF + c0 + c1 * g.sy + c2 * g.sz;
}

// wrap a padded coordinate into 1..N in a periodic direction (one period at most)
__host__ __device__ __forceinline__ int wrapc(int c, int N, int per)
{
    if (per) {
        if (c < 1) c += N;
        else if (c > N) c -= N;
    }
    return c;
}

// Per-level PCG scalars and the other device-resident scalars of a simulation.  They stay
// on the device: no dot product ever returns to the host (the paper's implementation copies
// each one back).
struct PcgScal {
    double rho, gamma, alpha, beta, rho0;
    double rsum;    // sum of r over the coupled cells (iD != 0), left by the kernel that last wrote r (R-T2)
    double nlive;   // number of coupled cells of the level (k_diag_flags)
    int live;   // 0 once a guard of DESIGN.md R-T has fired: later kernels of this smoother call are no-ops
    int stop_k; // one-sweep form (wl_pcgfused.cu): the iteration whose stopping criterion fired with its update still owed (0: none)
};

// time-dependent state of the map of one primitive of the body: xi = s .* (x - c)  (k_set_time)
struct PartState {
    double c[3];         // centre at the time the body was last placed
    double s[3];         // diagonal of the map
    double cdot[3];      // dc/dt
    double sdot_s[3];    // (ds/dt) / s
};

struct DevScal {
    PcgScal pcg[WL_MAXLEV];
    double t;            // time at which the body was last placed (measure!)
    double t_step;       // simulation time advanced by wl_step (never touched by wl_measure / wl_pressure_force)
    PartState part[4];   // the primitives of the body at time t
    PartState part_f[4]; // ... at the time the pressure-force integral is taken at
    float  vel[3];       // body velocity V (rigid translation: uniform)
    float  dt;           // time step of the running step
    float  dt_next;      // CFL result
    float  exit_corr;    // convective-exit mass correction
    float  pscale;       // w*dt of the running projection
    double cfl_max;
    double force[3];
    double resmax;
    int    nan_flag;
    int    band_count[4];// faces with mu1 != 0 found by the last measure!, per velocity component (each may exceed its third of the list)
    double energy[2];    // kinetic energy, enstrophy (wl_energy)
};

// reduction scratch: partial sums of up to 4 values per block + the arrival counter
struct CellBox { int lo[3], hi[3]; };     // inclusive range of cell coordinates (both 0 in an unused direction)

struct RedBuf {
    double* partial;     // [4][WL_MAX_PARTIALS]
    unsigned int* counter;
};

// ---- tiles: a kernel walks 32 x TY x TZ tiles, tile t = blockIdx.x, += gridDim.x -------
struct Tiling {
    int ntx, nty, ntz, ntiles;
    int o[3];     // origin (first coordinate) per direction
    int e[3];     // extent (number of cells) per direction
};

__device__ __forceinline__ bool tile_cell(const Tiling& T, int tile, int& c0, int& c1, int& c2)
{
    int tx = tile % T.ntx;
    int rem = tile / T.ntx;
    int ty = rem % T.nty;
    int tz = rem / T.nty;
    int i0 = tx * blockDim.x + threadIdx.x;
    int i1 = ty * blockDim.y + threadIdx.y;
    int i2 = tz * blockDim.z + threadIdx.z;
    c0 = T.o[0] + i0; c1 = T.o[1] + i1; c2 = T.o[2] + i2;
    return i0 < T.e[0] && i1 < T.e[1] && i2 < T.e[2];
}

// ---- deterministic reductions -----------------------------------------------------------
// Warp shuffle -> shared memory -> one partial per block -> the last block to arrive adds the
// partials in a fixed order.  The result is bit-reproducible run to run for a given grid size.
struct OpSum { __device__ static double f(double a, double b) { return a + b; } __device__ static double id() { return 0.0; } };
struct OpMax { __device__ static double f(double a, double b) { return a > b ? a : b; } __device__ static double id() { return -1e300; } };

template <class Op>
__device__ __forceinline__ double warp_red(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = Op::f(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Block-wide reduce of NV values; afterwards every thread of the LAST block to finish holds
// the grid totals in v[] and the function returns true there (false elsewhere).
template <int NV, class Op>
__device__ __forceinline__ bool grid_reduce(double (&v)[NV], const RedBuf& rb)
{
    __shared__ double sm[NV][32];
    __shared__ bool is_last;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nth = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, wid = tid >> 5, nw = (nth + 31) >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double w = warp_red<Op>(v[k]);
        if (lane == 0) sm[k][wid] = w;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double w = lane < nw ? sm[k][lane] : Op::id();
            w = warp_red<Op>(w);
            if (lane == 0) rb.partial[k * WL_MAX_PARTIALS + blockIdx.x] = w;
        }
        if (lane == 0) {
            __threadfence();
            unsigned int ticket = atomicAdd(rb.counter, 1u);
            is_last = (ticket == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    // fixed-order sum of the partials: thread-strided, then the same tree as above
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double w = Op::id();
        for (int b = tid; b < (int)gridDim.x; b += nth) w = Op::f(w, __ldcg(&rb.partial[k * WL_MAX_PARTIALS + b]));
        w = warp_red<Op>(w);
        if (lane == 0) sm[k][wid] = w;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double w = Op::id();
        for (int i = 0; i < nw; ++i) w = Op::f(w, sm[k][i]);
        v[k] = w;
    }
    if (tid == 0) *rb.counter = 0u;
    return true;
}
