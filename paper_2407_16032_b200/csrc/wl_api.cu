// wl_api.cu -- host side of libwl: workspace layout, the mom_step sequence, and the C ABI of
// include/wl.h.  No torch types; plain pointers and sizes only.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <new>
#include <nvtx3/nvToolsExt.h>
#include "wl_internal.h"
#include "wl_tma.cuh"

// NVTX range per routine of the paper's step (P:139 names them; the paper profiles with NVTX ranges under Nsight
// Systems): visible in nsys / ncu --nvtx, a no-op (one predicted branch) when no tool is attached.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};


// ------------------------------------------------------------------ launch geometry
dim3 wl_block(int nd) { return nd == 3 ? dim3(32, 4, 4) : dim3(32, 16, 1); }

Tiling wl_tiling(int nd, const int o[3], const int e[3])
{
    dim3 b = wl_block(nd);
    Tiling T;
    for (int d = 0; d < 3; ++d) { T.o[d] = o[d]; T.e[d] = e[d]; }
    T.ntx = (e[0] + b.x - 1) / b.x;
    T.nty = (e[1] + b.y - 1) / b.y;
    T.ntz = (e[2] + b.z - 1) / b.z;
    T.ntiles = T.ntx * T.nty * T.ntz;
    return T;
}
Tiling wl_tiles_interior(const wl_sim* s, const Grid& g)
{
    int o[3] = { 1, 1, s->nd == 3 ? 1 : 0 };
    int e[3] = { g.n[0], g.n[1], s->nd == 3 ? g.n[2] : 1 };
    return wl_tiling(s->nd, o, e);
}
Tiling wl_tiles_padded(const wl_sim* s, const Grid& g)
{
    int o[3] = { 0, 0, 0 };
    int e[3] = { g.S[0], g.S[1], g.S[2] };
    return wl_tiling(s->nd, o, e);
}
int wl_grid(const wl_sim* s, const Tiling& T)
{
    int cap = s->sm_count * 4;
    if (cap > WL_MAX_PARTIALS) cap = WL_MAX_PARTIALS;
    return T.ntiles < cap ? (T.ntiles > 0 ? T.ntiles : 1) : cap;
}
int wl_vgrid(const wl_sim* s, const VT& vt)
{
    int cap = s->sm_count * 4;
    if (cap > WL_MAX_PARTIALS) cap = WL_MAX_PARTIALS;
    return vt.ntiles < cap ? (vt.ntiles > 0 ? vt.ntiles : 1) : cap;
}
FlowP wl_flowp(const wl_sim* s)
{
    FlowP P;
    P.g = s->lev[0].g;
    P.nu = s->cfg.nu;
    for (int k = 0; k < 3; ++k) P.U[k] = s->cfg.U[k];
    P.exit_bc = s->cfg.exit_bc;
    P.Vf = s->Vf;
    return P;
}

// ------------------------------------------------------------------ config / layout
static int config_ok(const wl_config* c)
{
    if (!c) return 0;
    if (c->ndim != 2 && c->ndim != 3) return 0;
    for (int d = 0; d < c->ndim; ++d) if (c->dims[d] < 4 || c->dims[d] > 16384) return 0;
    if (!(c->nu >= 0.0f) || !(c->eps > 0.0f)) return 0;
    if (c->nextra < 0 || c->nextra > WL_MAX_EXTRA || (c->nextra > 0 && c->body.kind == WL_BODY_NONE)) return 0;
    for (int e = -1; e < c->nextra; ++e) {
        const wl_body& b = e < 0 ? c->body : c->extra[e];
        if (b.kind < (e < 0 ? 0 : 1) || b.kind > 4) return 0;
        if ((b.kind == WL_BODY_TORUS || b.kind == WL_BODY_CYLINDER) && (c->ndim != 3 || b.axis < 0 || b.axis > 2)) return 0;
        if (b.kind == WL_BODY_PLANE && (b.axis < 0 || b.axis >= c->ndim)) return 0;
        if (b.motion < 0 || b.motion > 1) return 0;
        if (e >= 0 && (c->extra_op[e] < 0 || c->extra_op[e] > 1)) return 0;
        for (int d = 0; d < 3; ++d) if (!(fabsf(b.scale_amp[d]) < 0.9f)) return 0;     // the map must stay invertible
    }
    if (c->tune.zc < 0 || c->tune.zc > 64 || c->tune.pk_blocks_per_sm < 0) return 0;
    if (c->precision < 0 || c->precision > 1 || c->tangent_param < 0 || c->tangent_param > WL_SEED_CENTRE) return 0;
    if (c->tangent_index < 0 || c->tangent_index > WL_MAX_EXTRA) return 0;
    if (c->exit_bc && c->periodic[0]) return 0;
    if (c->mg.smooth_iters < 1) return 0;
    return 1;
}

// the body velocity is a field rather than three scalars: several primitives, a non-rigid map, or spin (R-E3)
static int body_general(const wl_config* c)
{
    if (c->body.kind == WL_BODY_NONE) return 0;
    if (c->nextra > 0) return 1;
    const wl_body& b = c->body;
    return b.scale_amp[0] != 0.0f || b.scale_amp[1] != 0.0f || b.scale_amp[2] != 0.0f || b.spin != 0.0f;
}

static Grid make_grid(int nd, const int* n, const int* per)
{
    Grid g;
    for (int d = 0; d < 3; ++d) {
        g.n[d] = d < nd ? n[d] : 1;
        g.S[d] = d < nd ? n[d] + 2 : 1;
        g.per[d] = d < nd ? (per[d] ? 1 : 0) : 0;
    }
    // offset 7 + c0 of the last float4 group (and of its +4 neighbour) stays inside the row
    g.P = ((g.n[0] + 12 + 7) / 8) * 8;
    g.sy = g.P;
    g.sz = nd == 3 ? (int64_t)g.P * g.S[1] : 0;
    int64_t tot = (int64_t)g.P * g.S[1] * g.S[2];
    g.nalloc = ((tot + 63) / 64) * 64;
    return g;
}

#ifndef WL_PK_MIN_TILES
#define WL_PK_MIN_TILES 256     // the persistent-kernel levels take fewer planes per tile until they have this many tiles
#endif
// levels with at most this many cells run inside the persistent coarse-level kernels (k_coarse / k_tiny)
static long long pk_max_cells(const wl_config* c)
{
    if (c->tune.pk_max_cells < 0) return 0;
    return c->tune.pk_max_cells > 0 ? c->tune.pk_max_cells : (1ll << 20);     // 1 Mi: a 64 x 64 x 256 level (N2) is still one of them
}

// Vector tiling of a level.  Coarse levels are latency-bound, not bandwidth-bound: they take fewer
// planes per tile so that enough tiles (>= 4 per SM of a 148-SM B200 where the level allows) are in flight.
static VT make_vt(const wl_config* c, int nd, const Grid& g, int level)
{
    VT t;
    t.ngx = (g.n[0] + 3) / 4;
    t.lxl = 0;
    while ((1 << t.lxl) < t.ngx && t.lxl < 5) ++t.lxl;
    const int lx = 1 << t.lxl, ly = WL_VB >> t.lxl;
    t.ntx = (t.ngx + lx - 1) / lx;
    t.nty = (g.n[1] + ly - 1) / ly;
    const int zc0 = c->tune.zc > 0 ? c->tune.zc : 8;      // planes per tile
    t.zc = nd == 3 ? (g.n[2] < zc0 ? g.n[2] : zc0) : 1;
    if (level > 0 && (long long)g.n[0] * g.n[1] * g.n[2] <= pk_max_cells(c))
        while (t.zc > 1 && (int64_t)t.ntx * t.nty * ((g.n[2] + t.zc - 1) / t.zc) < WL_PK_MIN_TILES) t.zc = (t.zc + 1) / 2;
    t.ntz = nd == 3 ? (g.n[2] + t.zc - 1) / t.zc : 1;
    t.ntiles = t.ntx * t.nty * t.ntz;
    return t;
}

static int level_dims(const wl_config* c, int dims[WL_MAXLEV][3])
{
    int nd = c->ndim, n[3] = { c->dims[0], c->dims[1], nd == 3 ? c->dims[2] : 1 };
    int cap = c->mg.max_levels > 0 ? c->mg.max_levels : WL_MAXLEV;
    if (cap > WL_MAXLEV) cap = WL_MAXLEV;
    int nlev = 0;
    for (;;) {
        for (int d = 0; d < 3; ++d) dims[nlev][d] = n[d];
        ++nlev;
        if (nlev >= cap) break;
        int ok = 1;
        for (int d = 0; d < nd; ++d) if ((n[d] & 1) || n[d] <= 4) ok = 0;
        if (!ok) break;
        for (int d = 0; d < nd; ++d) n[d] /= 2;
    }
    return nlev;
}

struct Carver {
    char* base; size_t off;
    void* take(size_t bytes) { void* p = base ? base + off : nullptr; off += (bytes + 255) / 256 * 256; return p; }
};

// lays the arrays out in the workspace; with base == NULL only computes the size
static size_t layout(wl_sim* s, const wl_config* c, void* base)
{
    Carver cv = { (char*)base, 0 };
    int nd = c->ndim, dims[WL_MAXLEV][3];
    int nlev = level_dims(c, dims);
    DevScal* ds = (DevScal*)cv.take(sizeof(DevScal));
    double* partial = (double*)cv.take(sizeof(double) * 4 * WL_MAX_PARTIALS);
    unsigned int* counter = (unsigned int*)cv.take(256);
    LevDev* levdev = (LevDev*)cv.take(sizeof(LevDev) * WL_MAXLEV);
    double* pk_part = (double*)cv.take(sizeof(double) * 2 * 16 * WL_MAX_PARTIALS);    // room for slots of up to 16 doubles
    Grid g0 = make_grid(nd, dims[0], c->periodic);
    size_t sc = sizeof(float) * (size_t)g0.nalloc;
    float* ub[3];
    for (int k = 0; k < 3; ++k) ub[k] = (float*)cv.take(sc * nd);
    float* p = (float*)cv.take(sc);
    float* mu0 = (float*)cv.take(sc * nd);
    float* mu1 = (float*)cv.take(sc * nd * nd);
    float* Vf = body_general(c) ? (float*)cv.take(sc * nd) : nullptr;
    // band list: faces within eps of the body surface; a generous share of all faces (overflow falls back to a scan)
    int64_t ncell = (int64_t)dims[0][0] * dims[0][1] * dims[0][2];
    int64_t bcap = ncell * nd / 4;
    if (bcap < 4096) bcap = 4096;
    if (bcap > (1 << 26)) bcap = 1 << 26;
    if (c->body.kind == WL_BODY_NONE) bcap = 64;
    long long* band = (long long*)cv.take(sizeof(long long) * (size_t)bcap);
    if (s) {
        s->ds = ds; s->rb.partial = partial; s->rb.counter = counter;
        s->levdev = levdev; s->pk_part = pk_part;
        for (int k = 0; k < 3; ++k) s->ubuf[k] = ub[k];
        s->p = p; s->mu0 = mu0; s->mu1 = mu1; s->Vf = Vf;
        s->band_list = band; s->band_cap = (int)bcap;
        s->nlev = nlev; s->nd = nd;
    }
    for (int l = 0; l < nlev; ++l) {
        Grid g = make_grid(nd, dims[l], c->periodic);
        size_t scl = sizeof(float) * (size_t)g.nalloc;
        float* L = l == 0 ? mu0 : (float*)cv.take(scl * nd);
        float* iD = (float*)cv.take(scl);
        float* x = (float*)cv.take(scl);
        float* r = (float*)cv.take(scl);
        float* e = (float*)cv.take(scl);
        float* e2 = (float*)cv.take(scl);
        float* q = (float*)cv.take(scl);
        VT vt = make_vt(c, nd, g, l);
        // the one-sweep PCG form (wl_pcgfused.cu) ping-pongs r and q: two more arrays on the levels that take it.  Level 0
        // borrows them from the velocity buffer that is dead during the projection (solver_scratch()).
        const bool fused = wl_pcg_fused_shape(nd, g, vt) && (l == 0 || (long long)g.n[0] * g.n[1] * g.n[2] > pk_max_cells(c));
        float* r2 = fused && l > 0 ? (float*)cv.take(scl) : nullptr;
        float* q2 = fused && l > 0 ? (float*)cv.take(scl) : nullptr;
        if (s && l == 0) s->fused0 = fused ? 1 : 0;
        int* plain = (int*)cv.take(sizeof(int) * (size_t)vt.ntiles);
        int* uniform = (int*)cv.take(sizeof(int) * (size_t)vt.ntiles);
        int* tile_live = (int*)cv.take(sizeof(int) * (size_t)vt.ntiles);
        int* sched = fused ? (int*)cv.take(sizeof(int) * (size_t)vt.ntiles) : nullptr;
        if (s) {
            Level& lv = s->lev[l];
            lv.g = g; lv.L = L; lv.iD = iD; lv.x = x; lv.r = r; lv.e = e; lv.e2 = e2; lv.q = q; lv.r2 = r2; lv.q2 = q2;
            lv.vt = vt; lv.plain = plain; lv.uniform = uniform; lv.tile_live = tile_live; lv.sched = sched;
            lv.Lc = nd == 3 ? (float)(1 << l) : 1.0f;
            lv.iDc = 1.0f / (-(2.0f * nd) * lv.Lc);
        }
    }
    return cv.off;
}

static int is_generic(const wl_config* c) { return c->precision == 1 || c->tangent_param != WL_SEED_NONE; }

extern "C" size_t wl_workspace_bytes(const wl_config* cfg)
{
    if (!config_ok(cfg)) return 0;
    if (is_generic(cfg)) return wl_gen_bytes(cfg);
    return layout(nullptr, cfg, nullptr);
}

extern "C" int wl_abi_version(void) { return 2; }

// ------------------------------------------------------------------ the step
static void bc_all(wl_sim* s, float* u) { wl_k_bc(s, u); }

// defer_x: the caller runs apply_gradient next and nothing else reads x (the last smoother call may leave its final update to it)
static int solve(wl_sim* s, bool defer_x)
{
    const wl_mg& mg = s->cfg.mg;
    int nv = 0;
    if (mg.fixed_vcycles > 0) {
        for (; nv < mg.fixed_vcycles; ++nv) { wl_k_vcycle(s, 0); wl_k_smooth(s, 0, mg.smooth_iters, nv + 1 < mg.fixed_vcycles ? (s->nlev > 1 ? 2 : 1) : (defer_x ? -1 : 0)); }
        s->res[s->solve_slot] = -1.0;
    } else {
        double res = 0.0;
        for (;;) {
            wl_k_resmax(s);
            cudaMemcpyAsync(&s->hs->resmax, &s->ds->resmax, sizeof(double), cudaMemcpyDeviceToHost, s->st);
            if (cudaStreamSynchronize(s->st) != cudaSuccess) return WL_ECUDA;
            res = s->hs->resmax;
            if (!(res > (double)mg.tol) || nv >= mg.max_vcycles) break;
            wl_k_vcycle(s, 0);
            wl_k_smooth(s, 0, mg.smooth_iters);
            ++nv;
        }
        s->res[s->solve_slot] = res;
        if (res > (double)mg.tol) { s->noconv = 1; s->noconv_total++; }
    }
    s->vcycles[s->solve_slot] = nv;
    return WL_OK;
}

// Two level-0 scalar arrays the solver may scribble on: the first two components of a velocity buffer whose content is dead
// while `u` is being projected.  In mom_step the predictor's projection runs before ut is written, and the corrector's
// (u == ut) after the last use of u0; their ghost cells hold boundary values, which the stencil multiplies by the zero
// coefficient of a boundary face.
static void solver_scratch(wl_sim* s, const float* u)
{
    if (!s->fused0) return;
    float* b = (u == s->ut) ? s->u0 : s->ut;
    s->lev[0].r2 = b;
    s->lev[0].q2 = b + s->lev[0].g.nalloc;
}

// project!: z = div u; x = (w dt) p; solve A x = z; u -= L grad x; p = x/(w dt)
static int project(wl_sim* s, float* u, float w)
{
    NvtxRange nv("project!");
    solver_scratch(s, u);
    wl_k_residual(s, u, w);
    int rc = solve(s, true);
    wl_k_apply_gradient(s, u);
    return rc;
}

// mom_step (reading R-K/R-L).  ds->dt must hold the step's dt.
static int mom_step_body(wl_sim* s)
{
    // u0 <- u by swapping roles; the predictor writes the other buffer
    NvtxRange nv("mom_step!");
    float* t = s->u0; s->u0 = s->u; s->u = t;
    { NvtxRange r("conv_diff! + BDIM! (predictor)"); wl_k_conv_diff_bdim(s, s->u0, s->u0, s->u, 0); }
    { NvtxRange r("BC!"); bc_all(s, s->u); }
    if (s->cfg.exit_bc) { NvtxRange r("exitBC!"); wl_k_exit_bc(s, s->u, s->u0); }
    s->solve_slot = 0;
    int rc = project(s, s->u, 1.0f);
    if (rc != WL_OK) return rc;
    { NvtxRange r("BC!"); bc_all(s, s->u); }
    { NvtxRange r("conv_diff! + BDIM! + scale_u! (corrector)"); wl_k_conv_diff_bdim(s, s->u, s->u0, s->ut, 1); }
    { NvtxRange r("BC!"); bc_all(s, s->ut); }
    s->solve_slot = 1;
    rc = project(s, s->ut, 0.5f);
    if (rc != WL_OK) return rc;
    bc_all(s, s->ut);
    t = s->u; s->u = s->ut; s->ut = t;
    return WL_OK;
}

static int check(wl_sim* s)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(s->err, sizeof(s->err), "CUDA: %s", cudaGetErrorString(e));
        return WL_ECUDA;
    }
    return WL_OK;
}
static int sync(wl_sim* s)
{
    cudaError_t e = cudaStreamSynchronize(s->st);
    if (e != cudaSuccess) {
        snprintf(s->err, sizeof(s->err), "CUDA: %s", cudaGetErrorString(e));
        return WL_ECUDA;
    }
    return check(s);
}

// ------------------------------------------------------------------ C ABI
extern "C" int wl_sim_create(const wl_config* cfg, void* dev_ws, size_t ws_bytes, void* cuda_stream, wl_sim** out)
{
    if (!out) return WL_EINVAL;
    *out = nullptr;
    if (!config_ok(cfg)) return WL_EINVAL;
    size_t need = is_generic(cfg) ? wl_gen_bytes(cfg) : layout(nullptr, cfg, nullptr);
    if (!dev_ws || ws_bytes < need || ((uintptr_t)dev_ws & 255u)) return WL_ENOMEM;
    wl_sim* s = new (std::nothrow) wl_sim();     // value-initialised: every POD member zero
    if (!s) return WL_ENOMEM;
    s->cfg = *cfg;
    s->st = (cudaStream_t)cuda_stream;
    if (is_generic(cfg)) {                       // fp64 / tangent: the generic engine owns the workspace
        if (cudaMallocHost((void**)&s->hs, sizeof(DevScal)) != cudaSuccess) { delete s; return WL_ECUDA; }
        memset(s->hs, 0, sizeof(DevScal));
        int rc = wl_gen_create(s, dev_ws);
        if (rc != WL_OK) { cudaFreeHost(s->hs); delete s; return rc; }
        s->gen_dt_next = cfg->dt0;
        *out = s;
        return WL_OK;
    }
    layout(s, cfg, dev_ws);
    s->u = s->ubuf[0]; s->u0 = s->ubuf[1]; s->ut = s->ubuf[2];
    solver_scratch(s, s->u);
    {   // levels that run inside the persistent coarse-level kernel: from the first level >= 1 small enough
        const long long maxc = pk_max_cells(cfg);
        s->pk_level = s->nlev;
        for (int l = s->nlev - 1; l >= 1; --l) {
            const Grid& g = s->lev[l].g;
            if ((long long)g.n[0] * g.n[1] * g.n[2] <= maxc) s->pk_level = l; else break;
        }
    }
    s->tmc = new (std::nothrow) TmCache();
    if (!s->tmc) { delete s; return WL_ENOMEM; }
    s->tmc->n = 0;
    s->fast_A = !cfg->tune.no_fast_a;
    s->fused = !cfg->tune.no_fused;
    s->tiny_on = !cfg->tune.no_block_levels;
    s->small_cmax = -1;
    s->bulk_A = !cfg->tune.no_bulk;
    s->tma_cd = !cfg->tune.no_tma_cd;
    s->body.n = cfg->body.kind == WL_BODY_NONE ? 0 : 1 + cfg->nextra;
    s->body.eps = cfg->eps;
    s->body.general = body_general(cfg);
    for (int e = 0; e < s->body.n; ++e) {
        const wl_body& b = e == 0 ? cfg->body : cfg->extra[e - 1];
        PartP& q = s->body.part[e];
        q.kind = b.kind; q.axis = b.axis; q.R = b.R; q.r = b.r; q.shell = b.shell; q.spin = b.spin;
        q.scaled = b.scale_amp[0] != 0.0f || b.scale_amp[1] != 0.0f || b.scale_amp[2] != 0.0f;
        q.op = e == 0 ? 0 : cfg->extra_op[e - 1];
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        delete s;
        return WL_ECUDA;
    }
    s->sm_count = prop.multiProcessorCount;
    if (cudaMallocHost((void**)&s->hs, sizeof(DevScal)) != cudaSuccess) { delete s; return WL_ECUDA; }
    memset(s->hs, 0, sizeof(DevScal));
    if (cudaMemsetAsync(dev_ws, 0, need, s->st) != cudaSuccess) { cudaFreeHost(s->hs); delete s; return WL_ECUDA; }
    LevDev hl[WL_MAXLEV];
    memset(hl, 0, sizeof(hl));
    for (int l = 0; l < s->nlev; ++l) {
        const Level& lv = s->lev[l];
        LevDev& d = hl[l];
        d.g = lv.g; d.vt = lv.vt; d.L = lv.L; d.iD = lv.iD; d.x = lv.x; d.r = lv.r; d.e = lv.e; d.e2 = lv.e2; d.q = lv.q;
        d.plain = lv.plain; d.Lc = lv.Lc; d.iDc = lv.iDc;
    }
    if (cudaMemcpyAsync(s->levdev, hl, sizeof(hl), cudaMemcpyHostToDevice, s->st) != cudaSuccess) { cudaFreeHost(s->hs); delete s; return WL_ECUDA; }
    // initial state (R-V): u = U everywhere (all three buffers, so the exit plane is defined), p = 0, measure(0)
    for (int k = 0; k < 3; ++k) wl_k_fill_u(s, s->ubuf[k]);
    wl_k_set_time(s, 0.0, cfg->dt0, 2, 1);
    wl_k_measure(s);
    bc_all(s, s->u);
    int rc = sync(s);
    if (rc != WL_OK) { cudaFreeHost(s->hs); delete s; return rc; }
    *out = s;
    return WL_OK;
}

extern "C" int wl_sim_destroy(wl_sim* s)
{
    if (!s) return WL_EINVAL;
    cudaStreamSynchronize(s->st);
    wl_gen_destroy(s);
    delete s->tmc;
    if (s->hs) cudaFreeHost(s->hs);
    for (ProfRec& r : s->prof_recs) s->prof_pool.push_back(r);
    for (ProfRec& r : s->prof_pool) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    delete s;
    return WL_OK;
}

extern "C" const char* wl_last_error(const wl_sim* s) { return s ? s->err : "null handle"; }

static int64_t interior_count(const Grid& g) { return (int64_t)g.n[0] * g.n[1] * g.n[2]; }

// copy `ncomp` padded arrays out to an interior-sized user buffer, one component at a time
static int copy_out(wl_sim* s, const Grid& g, const float* padded, int ncomp, float* dst, int on_device, int whole = 0)
{
    int64_t ni = whole ? (int64_t)g.S[0] * g.S[1] * g.S[2] : interior_count(g);
    for (int m = 0; m < ncomp; ++m) {
        if (on_device) {
            wl_k_pack(s, g, padded + m * g.nalloc, dst + m * ni, 1, 1.0f, whole);
        } else {
            // staging: the level-0 q array (>= any interior size); it is scratch between solver calls
            float* stage = s->lev[0].q;
            wl_k_pack(s, g, padded + m * g.nalloc, stage, 1, 1.0f, whole);
            WL_CUDA_CHECK(s, cudaMemcpyAsync(dst + m * ni, stage, sizeof(float) * ni, cudaMemcpyDeviceToHost, s->st));
            WL_CUDA_CHECK(s, cudaStreamSynchronize(s->st));
        }
    }
    return check(s);
}
static int copy_in(wl_sim* s, const Grid& g, float* padded, int ncomp, const float* src, int on_device)
{
    int64_t ni = interior_count(g);
    for (int m = 0; m < ncomp; ++m) {
        if (on_device) {
            wl_k_unpack(s, g, src + m * ni, padded + m * g.nalloc, 1);
        } else {
            float* stage = s->lev[0].q;
            WL_CUDA_CHECK(s, cudaMemcpyAsync(stage, src + m * ni, sizeof(float) * ni, cudaMemcpyHostToDevice, s->st));
            wl_k_unpack(s, g, stage, padded + m * g.nalloc, 1);
            WL_CUDA_CHECK(s, cudaStreamSynchronize(s->st));
        }
    }
    return check(s);
}

extern "C" int wl_set_fields(wl_sim* s, const float* u, const float* p, int on_device)
{
    if (s && s->gen) return wl_gen_set_fields(s, u, p, on_device);
    if (!s) return WL_EINVAL;
    const Grid& g = s->lev[0].g;
    int rc;
    if (u) {
        if ((rc = copy_in(s, g, s->u, s->nd, u, on_device)) != WL_OK) return rc;
        bc_all(s, s->u);
    }
    if (p && (rc = copy_in(s, g, s->p, 1, p, on_device)) != WL_OK) return rc;
    return on_device ? check(s) : sync(s);
}

extern "C" int wl_get_fields(wl_sim* s, float* u, float* p, float* mu0, int on_device)
{
    if (s && s->gen) return wl_gen_get_fields(s, u, p, mu0, on_device);
    if (!s) return WL_EINVAL;
    const Grid& g = s->lev[0].g;
    int rc;
    if (u && (rc = copy_out(s, g, s->u, s->nd, u, on_device)) != WL_OK) return rc;
    if (p && (rc = copy_out(s, g, s->p, 1, p, on_device)) != WL_OK) return rc;
    if (mu0 && (rc = copy_out(s, g, s->mu0, s->nd, mu0, on_device)) != WL_OK) return rc;
    return on_device ? check(s) : sync(s);
}

extern "C" int wl_init_tgv(wl_sim* s, int sign)
{
    if (s && s->gen) return wl_gen_init_tgv(s, sign >= 0 ? 1 : -1);
    if (!s) return WL_EINVAL;
    wl_k_init_tgv(s, sign >= 0 ? 1 : -1);
    bc_all(s, s->u);
    return check(s);
}

extern "C" int wl_measure(wl_sim* s, double t)
{
    if (s && s->gen) { s->gen_tbody = t; return wl_gen_measure(s, t); }
    if (!s) return WL_EINVAL;
    NvtxRange r("measure!");
    wl_k_set_time(s, t, 0.0f, 1, -1);
    wl_k_measure(s);
    return check(s);
}

extern "C" int wl_mom_step(wl_sim* s, float dt)
{
    if (s && s->gen) return dt > 0.0f ? wl_gen_mom_step(s, (double)dt) : WL_EINVAL;
    if (!s || !(dt > 0.0f)) return WL_EINVAL;
    wl_k_set_time(s, 0.0, dt, -1, 1);
    int rc = mom_step_body(s);
    if (rc != WL_OK) return rc;
    return check(s);
}

extern "C" int wl_step(wl_sim* s, double t, float dt, int adaptive)
{
    if (s && s->gen) {                           // generic engine: the CFL result makes a host round trip
        const int dev = adaptive && s->primed;
        if (!dev && !(dt > 0.0f)) return WL_EINVAL;
        const float dtu = dev ? s->gen_dt_next : dt;
        const double tu = dev ? s->gen_t + (double)dtu : t;
        int rc = WL_OK;
        if (s->cfg.body.kind != WL_BODY_NONE && (s->cfg.body.motion != WL_MOTION_STATIC || s->cfg.nextra > 0 || s->cfg.body.scale_freq != 0.0f)) {
            s->gen_tbody = tu;
            rc = wl_gen_measure(s, tu);
        }
        if (rc == WL_OK) rc = wl_gen_mom_step(s, (double)dtu);
        if (rc == WL_OK) rc = wl_gen_cfl(s, &s->gen_dt_next);
        s->gen_t = tu;
        s->primed = adaptive ? 1 : 0;
        return rc;
    }
    if (!s) return WL_EINVAL;
    int dev = adaptive && s->primed;   // device-resident t and dt are valid
    if (!dev && !(dt > 0.0f)) return WL_EINVAL;
    wl_k_set_time(s, t, dt, dev ? 0 : 2, dev ? 0 : 1);
    if (s->cfg.body.kind != WL_BODY_NONE && s->cfg.body.motion != WL_MOTION_STATIC) { NvtxRange r("measure!"); wl_k_measure(s); }
    int rc = mom_step_body(s);
    if (rc != WL_OK) return rc;
    { NvtxRange r("CFL!"); wl_k_cfl(s, s->u); }
    s->primed = adaptive ? 1 : 0;
    return check(s);
}

extern "C" int wl_cfl(wl_sim* s, float* dt_out)
{
    if (s && s->gen && dt_out) {
        int rc = wl_gen_cfl(s, dt_out);
        if (rc == WL_OK && s->noconv) { s->noconv = 0; return WL_ENOCONV; }
        return rc;
    }
    if (!s || !dt_out) return WL_EINVAL;
    wl_k_cfl(s, s->u);
    WL_CUDA_CHECK(s, cudaMemcpyAsync(&s->hs->dt_next, &s->ds->dt_next, sizeof(float), cudaMemcpyDeviceToHost, s->st));
    WL_CUDA_CHECK(s, cudaMemcpyAsync(&s->hs->nan_flag, &s->ds->nan_flag, sizeof(int), cudaMemcpyDeviceToHost, s->st));
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    *dt_out = s->hs->dt_next;
    if (s->noconv) { s->noconv = 0; return WL_ENOCONV; }
    return WL_OK;
}

extern "C" int wl_pressure_force(wl_sim* s, double t, float F_out[3])
{
    if (s && s->gen && F_out) {
        double F[3];
        int rc = wl_gen_force(s, t == t ? t : s->gen_tbody, F, nullptr);
        for (int k = 0; k < 3; ++k) F_out[k] = (float)F[k];
        return rc;
    }
    if (!s || !F_out) return WL_EINVAL;
    wl_k_force(s, t);                                // NaN: the body where measure! last placed it
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->hs->force, s->ds->force, 3 * sizeof(double), cudaMemcpyDeviceToHost, s->st));
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    for (int k = 0; k < 3; ++k) F_out[k] = (float)s->hs->force[k];
    return WL_OK;
}

extern "C" int wl_energy(wl_sim* s, double out[2])
{
    if (s && s->gen && out) return wl_gen_energy(s, out, nullptr);
    if (!s || !out) return WL_EINVAL;
    wl_k_energy(s, s->u);
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->hs->energy, s->ds->energy, 2 * sizeof(double), cudaMemcpyDeviceToHost, s->st));
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    out[0] = s->hs->energy[0]; out[1] = s->hs->energy[1];
    return WL_OK;
}

// ---- fp64 / tangent views (generic engine)
extern "C" int wl_get_fields_f64(wl_sim* s, double* u, double* p, int tangent, int on_device)
{
    if (!s || !s->gen) return WL_EINVAL;
    return wl_gen_get_fields_f64(s, u, p, tangent ? 1 : 0, on_device);
}
extern "C" int wl_set_fields_f64(wl_sim* s, const double* u, const double* p, int on_device)
{
    if (!s || !s->gen) return WL_EINVAL;
    return wl_gen_set_fields_f64(s, u, p, on_device);
}
extern "C" int wl_pressure_force_f64(wl_sim* s, double t, double F[3], double dF[3])
{
    if (!s || !s->gen || !F) return WL_EINVAL;
    return wl_gen_force(s, t == t ? t : s->gen_tbody, F, dF);
}
extern "C" int wl_energy_f64(wl_sim* s, double out[2], double dout[2])
{
    if (!s || !s->gen || !out) return WL_EINVAL;
    return wl_gen_energy(s, out, dout);
}
extern "C" int wl_dbg_get_f64(wl_sim* s, const char* name, int level, int tangent, double* out, size_t out_doubles)
{
    if (!s || !s->gen || !name || !out) return WL_EINVAL;
    return wl_gen_dbg_get(s, name, level, tangent ? 1 : 0, out, out_doubles);
}

extern "C" int wl_stats(wl_sim* s, wl_stats_t* out)
{
    if (!s || !out) return WL_EINVAL;
    out->vcycles[0] = s->vcycles[0]; out->vcycles[1] = s->vcycles[1];
    out->res[0] = s->res[0]; out->res[1] = s->res[1];
    out->nlevels = s->nlev;
    out->kernel_launches = s->launches;
    out->nan_flag = s->hs->nan_flag;
    out->noconv = s->noconv_total;
    return WL_OK;
}

extern "C" int wl_level_dims(const wl_sim* s, int level, int dims_out[3])
{
    if (!s || level < 0 || level >= s->nlev) return WL_EINVAL;
    if (s->gen) { for (int d = 0; d < 3; ++d) dims_out[d] = d < s->nd ? s->cfg.dims[d] >> level : 1; return WL_OK; }
    for (int d = 0; d < 3; ++d) dims_out[d] = s->lev[level].g.n[d];
    return WL_OK;
}

// ---- per-kernel-class timing (CUDA events on the handle's stream)
static const char* const kern_names[WLK_COUNT] = {
    "set_time", "measure", "poisson_update", "conv_diff_bdim", "bc", "exit_bc", "residual", "restrict", "prolong",
    "pcg_init", "pcg_matvec", "pcg_update", "pcg_dir", "apply_gradient", "cfl", "force", "resmax", "misc", "conv_diff_band", "vcycle", "pcg_fused",
    "energy", "small_levels"
};

extern "C" int wl_prof_enable(wl_sim* s, int enable)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s) return WL_EINVAL;
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    for (ProfRec& r : s->prof_recs) s->prof_pool.push_back(r);
    s->prof_recs.clear();
    s->prof_on = enable ? 1 : 0;
    return WL_OK;
}

extern "C" int wl_prof_read(wl_sim* s, int cls, char* name_out, size_t name_bytes, double* ms_total, int* launches)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s || cls < 0) return WL_EINVAL;
    if (cls >= 2 * WLK_COUNT) return 1;
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    double ms = 0.0;
    int n = 0;
    for (const ProfRec& r : s->prof_recs) {
        if (r.cls != cls) continue;
        float t = 0.0f;
        WL_CUDA_CHECK(s, cudaEventElapsedTime(&t, r.a, r.b));
        ms += (double)t;
        ++n;
    }
    if (name_out && name_bytes) snprintf(name_out, name_bytes, "%s%s", kern_names[cls / 2], (cls & 1) ? ".coarse" : "");
    if (ms_total) *ms_total = ms;
    if (launches) *launches = n;
    return WL_OK;
}

// ---- stage hooks
extern "C" int wl_dbg_save_u0(wl_sim* s)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s) return WL_EINVAL;
    const Grid& g = s->lev[0].g;
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->u0, s->u, sizeof(float) * g.nalloc * s->nd, cudaMemcpyDeviceToDevice, s->st));
    return WL_OK;
}
extern "C" int wl_dbg_conv_diff_bdim(wl_sim* s, float dt, int corrector)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s) return WL_EINVAL;
    wl_k_set_time(s, 0.0, dt, -1, 1);
    wl_k_conv_diff_bdim(s, s->u, s->u0, s->ut, corrector);
    float* t = s->u; s->u = s->ut; s->ut = t;
    return check(s);
}
extern "C" int wl_dbg_bc(wl_sim* s) { if (!s || s->gen) return WL_EINVAL; bc_all(s, s->u); return check(s); }
extern "C" int wl_dbg_exit_bc(wl_sim* s, float dt)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s) return WL_EINVAL;
    wl_k_set_time(s, 0.0, dt, -1, 1);
    wl_k_exit_bc(s, s->u, s->u0);
    return check(s);
}
extern "C" int wl_dbg_project(wl_sim* s, float w, float dt)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s) return WL_EINVAL;
    wl_k_set_time(s, 0.0, dt, -1, 1);
    s->solve_slot = 0;
    int rc = project(s, s->u, w);
    return rc != WL_OK ? rc : check(s);
}
extern "C" int wl_dbg_residual(wl_sim* s)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    // r = div u - A x with the CURRENT x: expressed through k_residual by p := x, w dt := 1
    if (!s) return WL_EINVAL;
    const Grid& g = s->lev[0].g;
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->lev[0].q, s->p, sizeof(float) * g.nalloc, cudaMemcpyDeviceToDevice, s->st));
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->p, s->lev[0].x, sizeof(float) * g.nalloc, cudaMemcpyDeviceToDevice, s->st));
    wl_k_set_time(s, 0.0, 1.0f, -1, 1);
    wl_k_residual(s, s->u, 1.0f);
    WL_CUDA_CHECK(s, cudaMemcpyAsync(s->p, s->lev[0].q, sizeof(float) * g.nalloc, cudaMemcpyDeviceToDevice, s->st));
    return check(s);
}
extern "C" int wl_dbg_apply_gradient(wl_sim* s) { if (!s || s->gen) return WL_EINVAL; wl_k_apply_gradient(s, s->u); return check(s); }
extern "C" int wl_dbg_restrict(wl_sim* s, int l) { if (!s || s->gen || l < 0 || l + 1 >= s->nlev) return WL_EINVAL; wl_k_restrict(s, l); return check(s); }
extern "C" int wl_dbg_prolong(wl_sim* s, int l) { if (!s || s->gen || l < 0 || l + 1 >= s->nlev) return WL_EINVAL; wl_k_prolong(s, l); return check(s); }
extern "C" int wl_dbg_smooth(wl_sim* s, int l, int iters)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s || l < 0 || l >= s->nlev || iters < 1) return WL_EINVAL;
    wl_k_rsum(s, l);          // in a solve the kernel that wrote r leaves this sum
    wl_k_smooth(s, l, iters);
    return check(s);
}
extern "C" int wl_dbg_vcycle(wl_sim* s, int l) { if (!s || s->gen || l < 0 || l >= s->nlev) return WL_EINVAL; wl_k_vcycle(s, l); return check(s); }

// runs n coarse-level passes (kind: 0 restrict level->level+1, 1 smooth, 2 prolong level+1->level) as ONE k_coarse launch
extern "C" int wl_dbg_coarse_prog(wl_sim* s, int n, const int* kinds, const int* levels, const int* iters)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s || n < 1 || n > 3 * WL_MAXLEV || !kinds || !levels || !iters) return WL_EINVAL;
    CoarseProg P; P.n = n;
    for (int k = 0; k < n; ++k) {
        const int top = kinds[k] == COP_SMOOTH ? s->nlev - 1 : s->nlev - 2;
        if (kinds[k] < 0 || kinds[k] > 2 || levels[k] < 0 || levels[k] > top || (kinds[k] == COP_SMOOTH && iters[k] < 1)) return WL_EINVAL;
        P.op[k].kind = kinds[k]; P.op[k].level = levels[k]; P.op[k].iters = iters[k];
    }
    wl_k_coarse_prog(s, P);
    return check(s);
}

// PCG scalars of a level: rho, gamma, alpha, beta, rho0, rsum, nlive, live
extern "C" int wl_dbg_pcg_scalars(wl_sim* s, int level, double out[8])
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s || level < 0 || level >= s->nlev || !out) return WL_EINVAL;
    PcgScal h;
    WL_CUDA_CHECK(s, cudaMemcpyAsync(&h, &s->ds->pcg[level], sizeof(PcgScal), cudaMemcpyDeviceToHost, s->st));
    int rc = sync(s);
    if (rc != WL_OK) return rc;
    out[0] = h.rho; out[1] = h.gamma; out[2] = h.alpha; out[3] = h.beta; out[4] = h.rho0; out[5] = h.rsum; out[6] = h.nlive; out[7] = (double)h.live;
    return WL_OK;
}

static int find_array(wl_sim* s, const char* name, int level, float** arr, int* ncomp, const Grid** g)
{
    if (level < 0 || level >= s->nlev) return WL_EINVAL;
    Level& lv = s->lev[level];
    *g = &lv.g; *ncomp = 1;
    if (!strcmp(name, "L")) { *arr = lv.L; *ncomp = s->nd; return WL_OK; }
    if (!strcmp(name, "iD")) { *arr = lv.iD; return WL_OK; }
    if (!strcmp(name, "x")) { *arr = lv.x; return WL_OK; }
    if (!strcmp(name, "r")) { *arr = lv.r; return WL_OK; }
    if (!strcmp(name, "e")) { *arr = lv.e; return WL_OK; }
    if (!strcmp(name, "q")) { *arr = lv.q; return WL_OK; }
    *g = &s->lev[0].g;
    if (!strcmp(name, "u")) { *arr = s->u; *ncomp = s->nd; return WL_OK; }
    if (!strcmp(name, "u0")) { *arr = s->u0; *ncomp = s->nd; return WL_OK; }
    if (!strcmp(name, "p")) { *arr = s->p; return WL_OK; }
    if (!strcmp(name, "mu0")) { *arr = s->mu0; *ncomp = s->nd; return WL_OK; }
    if (!strcmp(name, "mu1")) { *arr = s->mu1; *ncomp = s->nd * s->nd; return WL_OK; }
    if (!strcmp(name, "V") && s->Vf) { *arr = s->Vf; *ncomp = s->nd; return WL_OK; }
    return WL_EINVAL;
}
static int dbg_get(wl_sim* s, const char* name, int level, float* out, size_t out_floats, int whole)
{
    if (!s || !name || !out || s->gen) return WL_EINVAL;
    float* arr; int nc; const Grid* g;
    int rc = find_array(s, name, level, &arr, &nc, &g);
    if (rc != WL_OK) return rc;
    int64_t cnt = whole ? (int64_t)g->S[0] * g->S[1] * g->S[2] : interior_count(*g);
    if (out_floats < (size_t)(cnt * nc)) return WL_EINVAL;
    if (arr == s->lev[0].q) {   // q is the staging buffer: go through e's slot is not possible; copy via ut
        WL_CUDA_CHECK(s, cudaMemcpyAsync(s->ut, arr, sizeof(float) * g->nalloc, cudaMemcpyDeviceToDevice, s->st));
        arr = s->ut;
    }
    rc = copy_out(s, *g, arr, nc, out, 0, whole);
    return rc != WL_OK ? rc : nc;
}
extern "C" int wl_dbg_get(wl_sim* s, const char* name, int level, float* out, size_t out_floats)
{
    return dbg_get(s, name, level, out, out_floats, 0);
}
extern "C" int wl_dbg_get_padded(wl_sim* s, const char* name, int level, float* out, size_t out_floats)
{
    return dbg_get(s, name, level, out, out_floats, 1);
}
extern "C" int wl_dbg_set(wl_sim* s, const char* name, int level, const float* in, size_t in_floats)
{
    if (s && s->gen) return WL_EINVAL;      // stage hooks belong to the tuned kernels
    if (!s || !name || !in) return WL_EINVAL;
    float* arr; int nc; const Grid* g;
    int rc = find_array(s, name, level, &arr, &nc, &g);
    if (rc != WL_OK) return rc;
    if (in_floats < (size_t)(interior_count(*g) * nc) || arr == s->lev[0].q) return WL_EINVAL;
    rc = copy_in(s, *g, arr, nc, in, 0);
    s->measured = 0;        // the next measure! takes nothing for unchanged
    return rc != WL_OK ? rc : nc;
}
