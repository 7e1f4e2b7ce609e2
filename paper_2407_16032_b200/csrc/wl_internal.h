// wl_internal.h -- host-side handle of libwl and the kernel-launch entry points shared by
// the translation units (wl_api.cu, wl_flow.cu, wl_convdiff.cu, wl_poisson.cu).
#pragma once
#include "../../include/wl.h"
#include "wl_common.cuh"
#include "wl_body.cuh"
#include "wl_vec.cuh"
#include <vector>

// kernel classes for launch accounting and the optional per-class CUDA-event timing (wl_prof_*)
enum WlKern {
    WLK_SET_TIME, WLK_MEASURE, WLK_POISSON_UPDATE, WLK_CONVDIFF, WLK_BC, WLK_EXIT_BC, WLK_RESIDUAL,
    WLK_RESTRICT, WLK_PROLONG, WLK_PCG_INIT, WLK_PCG_MATVEC, WLK_PCG_UPDATE, WLK_PCG_DIR,
    WLK_GRADIENT, WLK_CFL, WLK_FORCE, WLK_RESMAX, WLK_MISC, WLK_CONVDIFF_BAND, WLK_COARSE, WLK_PCG_FUSED, WLK_ENERGY, WLK_SMALL, WLK_COUNT
};
struct ProfRec { cudaEvent_t a, b; int cls; };

struct Level {
    Grid g;
    float* L;    // nd face-coefficient arrays (level 0: alias of mu0), stride g.nalloc
    float* iD;   // inverse diagonal
    float* x;    // solution / correction
    float* r;    // residual
    float* e;    // CG direction (ping)
    float* e2;   // CG direction (pong): pass A reads one and writes the other
    float* q;    // A e
    float* r2;   // second residual and A e buffers of the one-sweep PCG form (wl_pcgfused.cu); null on levels that do not take it
    float* q2;
    VT vt;       // vector tiling of this level
    int* sched;     // levels of the one-sweep smoother: the order its blocks take the tiles in (tile | mode << 24), TM_GEN tiles first (k_tile_sched)
    int* tile_live; // per tile: number of coupled cells (iD != 0) in it, kept so that k_diag_flags can skip tiles the body cannot reach
    int* uniform; // per-tile flag: every face coefficient of every cell of the tile equals Lc
    int* plain;  // per-tile flag: the tile and its face-neighbour tiles are uniform (kernels skip L and iD loads)
    float Lc;    // face coefficient of a body-free, boundary-free cell on this level (R-S: 1, or 2^l in 3-D)
    float iDc;   // 1 / (-2 n Lc)
};

// device-side copy of a level (array in the workspace, read by the persistent coarse-level kernel)
struct LevDev {
    Grid g; VT vt;
    float *L, *iD, *x, *r, *e, *e2, *q;
    int* plain;
    float Lc, iDc;
};

// a chain of coarse-level passes run by one k_coarse launch
enum { COP_RESTRICT = 0, COP_SMOOTH = 1, COP_PROLONG = 2 };   // RESTRICT: level -> level+1; PROLONG: level+1 -> level
struct CoarseOp { int kind, level, iters; };
struct CoarseProg { int n; CoarseOp op[3 * WL_MAXLEV]; };

struct wl_sim {
    wl_config cfg;
    int nd, nlev;
    Level lev[WL_MAXLEV];
    float* ubuf[3];          // three rotating velocity buffers (nd comps each)
    float *u, *u0, *ut;      // roles: current, start-of-step, scratch/next
    float* p;                // pressure (unscaled)
    float* mu0;              // nd comps
    float* mu1;              // nd*nd comps
    float* Vf;               // body velocity per face (nd comps) when the body is general (BodyP::general), else null: V is ds->vel
    long long* band_list;    // faces with mu1 != 0, written by measure!: (array offset << 2) | component
    int band_cap;            // capacity of band_list (entries)
    int cd_attr_set;         // dynamic shared-memory attributes set: bits 2, 4 conv_diff kernels, 16 k_pcg_fused
    DevScal* ds;             // device-resident scalars
    DevScal* hs;             // pinned host mirror for read-back
    RedBuf rb;
    LevDev* levdev;          // device array [nlev]
    double* pk_part;         // per-block partial sums of k_coarse
    int pk_level;            // levels >= pk_level run inside k_coarse (nlev: none)
    int pk_blocks;           // co-resident grid of k_coarse (0: not yet queried)
    int tiny_on;             // small levels run on chip in the one-cluster kernel k_small (wl_tuning.no_block_levels switches it off)
    int small_cmax;          // largest cluster k_small can be launched with on this device (-1: not yet queried, 0: none)
    int measured;            // measure! has run over the whole grid once: later calls only visit the box the body can reach
    int tma_cd;              // conv_diff from the TMA-fed ring (k_cd_tile3) where it applies (wl_tuning.no_tma_cd switches it off)
    int bulk_A;              // k_pcg_A_fast takes its operand planes as TMA boxes where it can (wl_tuning.no_bulk switches it off)
    int mbox_lo[3], mbox_hi[3]; // padded coordinates of the box the last measure! rewrote (the whole array the first time)
    const float* pend_e;     // the last smoother call of a solve left its final x += alpha e to apply_gradient (wl_pcgfused.cu): the direction, else null
    int pend_k;              // ... and the iteration whose update that is
    const float *pr_r, *pr_q, *pr_e;   // between two V-cycles of a solve: the smoother left x += alpha e, r -= alpha q to restrict(0) and prolong(0) (null: nothing pending)
    int pr_k;
    int fused0;              // level 0 takes the one-sweep PCG form; its r2, q2 live in a dead velocity buffer (wl_api.cu solver_scratch)
    int fused;               // PCG smoother in its one-sweep form where the level allows (wl_tuning.no_fused switches it off)
    int fast_A;              // uniform tiles of PCG pass A go through k_pcg_A_fast (wl_tuning.no_fast_a switches it off)
    BodyP body;
    cudaStream_t st;
    int launches;
    int vcycles[2];
    double res[2];
    int solve_slot;
    int noconv;              // a tolerance-mode solve hit max_vcycles since the last wl_cfl (which reports and clears it)
    int noconv_total;        // ... since create (wl_stats)
    int primed;              // device-resident t and dt are valid (adaptive wl_step)
    int sm_count;
    struct TmCache* tmc;     // encoded tensor maps of the solver and velocity arrays (wl_tma.cuh)
    void* gen;               // the generic engine (wl_generic.cu) when cfg.precision = 1 or a tangent is asked for, else null
    int gen_kind;            // 1: double, 2: dual
    double gen_t, gen_tbody; // simulation time / time the body was last placed (generic engine: host-side)
    float gen_dt_next;
    char err[256];
    // profiling (off by default): every launch bracketed by two events on the stream
    int prof_on;
    std::vector<ProfRec> prof_recs;      // records in use since the last read
    std::vector<ProfRec> prof_pool;      // events kept for reuse
};

// One kernel launch: counts it and, when profiling is on, brackets it with CUDA events.
// Class index = 2*kind + (coarse ? 1 : 0): multigrid levels > 0 are accounted separately.
struct ProfScope {
    wl_sim* s; cudaEvent_t stop; 
    ProfScope(wl_sim* s_, int kind, int coarse = 0) : s(s_), stop(nullptr)
    {
        s->launches++;
        if (!s->prof_on) return;
        ProfRec r;
        if (!s->prof_pool.empty()) { r = s->prof_pool.back(); s->prof_pool.pop_back(); }
        else { cudaEventCreate(&r.a); cudaEventCreate(&r.b); }
        r.cls = 2 * kind + (coarse ? 1 : 0);
        cudaEventRecord(r.a, s->st);
        stop = r.b;
        s->prof_recs.push_back(r);
    }
    ~ProfScope() { if (stop) cudaEventRecord(stop, s->st); }
};

// flow-side parameters passed by value to kernels
struct FlowP {
    Grid g;
    float nu;
    float U[3];
    int exit_bc;
    const float* Vf;   // body velocity per face (general bodies), or null: uniform V from DevScal
};

// launch geometry
dim3 wl_block(int nd);
Tiling wl_tiling(int nd, const int o[3], const int e[3]);
int wl_grid(const wl_sim* s, const Tiling& T);
int wl_vgrid(const wl_sim* s, const VT& vt);
Tiling wl_tiles_interior(const wl_sim* s, const Grid& g);
Tiling wl_tiles_padded(const wl_sim* s, const Grid& g);
FlowP wl_flowp(const wl_sim* s);

// wl_flow.cu
void wl_k_set_time(wl_sim* s, double t, float dt, int t_mode, int dt_mode);   // t: 2 host value, also the simulation time; 1 host value, body only; 0 device (t_step + dt); -1 keep.  dt: 1 host, 0 device, -1 keep
void wl_k_measure(wl_sim* s);
void wl_body_box(const wl_sim* s, float margin, int interior, int o[3], int e[3]);
void wl_k_bc(wl_sim* s, float* u);
void wl_k_exit_bc(wl_sim* s, float* u, const float* u0);
void wl_k_cfl(wl_sim* s, const float* u);
void wl_k_force(wl_sim* s, double t);                // t = NaN: the body where measure! last placed it
void wl_k_energy(wl_sim* s, const float* u);
void wl_k_init_tgv(wl_sim* s, int sign);
void wl_k_fill(wl_sim* s, float* a, int64_t n, float v);
void wl_k_fill_u(wl_sim* s, float* u);
void wl_k_pack(wl_sim* s, const Grid& g, const float* padded, float* dense, int ncomp, float scale, int whole);
void wl_k_unpack(wl_sim* s, const Grid& g, const float* interior, float* padded, int ncomp);
// wl_convdiff.cu
void wl_k_conv_diff_bdim(wl_sim* s, const float* w, const float* u0, float* out, int corrector);
// wl_pcgfast.cu
int wl_pcg_fast_ok(const wl_sim* s, int l);
void wl_k_pcg_A_fast(wl_sim* s, int l, int first, const float* ein, float* eout);
// wl_pcgfused.cu
int wl_pcg_fused_shape(int nd, const Grid& g, const VT& vt);    // the one-sweep form can take a level of this shape
int wl_k_smooth_fused(wl_sim* s, int l, int iters, int need_r);              // 0: not taken (the caller runs the two-pass form)
// wl_generic.cu
size_t wl_gen_bytes(const wl_config* c);
int wl_gen_create(wl_sim* s, void* ws);
void wl_gen_destroy(wl_sim* s);
int wl_gen_measure(wl_sim* s, double t);
int wl_gen_mom_step(wl_sim* s, double dt);
int wl_gen_cfl(wl_sim* s, float* dt_out);
int wl_gen_force(wl_sim* s, double t, double* F, double* dF);
int wl_gen_energy(wl_sim* s, double* out, double* dout);
int wl_gen_init_tgv(wl_sim* s, int sign);
int wl_gen_set_fields(wl_sim* s, const float* u, const float* p, int on_device);
int wl_gen_set_fields_f64(wl_sim* s, const double* u, const double* p, int on_device);
int wl_gen_get_fields(wl_sim* s, float* u, float* p, float* mu0, int on_device);
int wl_gen_get_fields_f64(wl_sim* s, double* u, double* p, int lane, int on_device);
int wl_gen_dbg_get(wl_sim* s, const char* name, int level, int lane, double* out, size_t n);
// wl_small.cu
int wl_small_max_cluster(wl_sim* s);
int wl_small_blocks(const Grid& g, int cmax);
int wl_k_small_prog(wl_sim* s, const CoarseProg& P, int C);
// wl_poisson.cu
void wl_k_poisson_update(wl_sim* s);                 // iD on level 0, coarse L and iD
void wl_k_residual(wl_sim* s, const float* u, float w);   // pscale = w*dt; x = pscale*p; r = div u - A x
void wl_k_restrict(wl_sim* s, int l);                // r_{l+1} = sum children r_l ; x_{l+1} = 0
void wl_k_prolong(wl_sim* s, int l);                 // x_l += P x_{l+1}; r_l -= A_l P x_{l+1}
// need_r = 0: nobody reads the residual of this level before it is rewritten (a coarse level before its prolongation, the
// last smoother call of a solve with a fixed number of V-cycles): the one-sweep form then leaves r one update behind
void wl_k_smooth(wl_sim* s, int l, int iters, int need_r = 1);   // need_r: 1 the residual is read afterwards; 0 only x; -1 only x, and by apply_gradient alone (level 0); 2 x and r, and by the restrict(0) / prolong(0) of the next V-cycle alone
void wl_k_coarse_prog(wl_sim* s, const CoarseProg& P);   // one k_coarse launch
void wl_k_rsum(wl_sim* s, int l);                    // pcg[l].rsum = sum of r over the coupled cells (stage hooks)
void wl_k_vcycle(wl_sim* s, int l);
void wl_k_apply_gradient(wl_sim* s, float* u);       // u -= L grad x ; p = x / pscale
void wl_k_resmax(wl_sim* s);                         // ds->resmax = max |r_0|

#define WL_CUDA_CHECK(s, call)                                                              \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            snprintf((s)->err, sizeof((s)->err), "%s:%d %s", __FILE__, __LINE__, cudaGetErrorString(e_)); \
            return WL_ECUDA;                                                                \
        }                                                                                   \
    } while (0)
