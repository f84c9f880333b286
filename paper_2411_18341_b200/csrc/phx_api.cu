// phx_api.cu -- the C ABI of libphx (include/phx.h): handle, validation, workspace carving, copies,
// canonical coefficients, launch plan (CUDA graphs of the per-step kernel sequence).
// There is no CPU path: every step of the method runs in the kernels of this library.
#include "../../include/phx.h"

#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "phx_adaptive.h"
#include "phx_launch.h"
#include "phx_stage.cuh"
#include "phx_step.cuh"

using namespace phx;

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
    size_t psi[2], ya[2], yb[2], acc[2], n[2], na[2], nb[2], nacc[2], V, P, E, step, total;
    size_t K[7][2], Kn[7][2], dpctl, dplog;   // adaptive integrator (PHX_INT_DP54 only)
    size_t scratch_bytes;   // yb[0], acc[0] are contiguous and dead between steps in every variant: scratch
};

bool desc_ok(const phx_grid_desc* d) {
    if (!d) return false;
    if (d->nx < 3 || d->ny < 3 || d->batch < 1 || d->batch > 65535) return false;
    if (!(d->dx > 0) || !(d->dy > 0)) return false;
    if (d->prec != PHX_C32 && d->prec != PHX_C64) return false;
    if (d->model < PHX_SCALAR || d->model > PHX_SPINOR_RESERVOIR) return false;
    if ((d->bc_x != 0 && d->bc_x != 1) || (d->bc_y != 0 && d->bc_y != 1)) return false;
    if (d->noise != 0 && d->noise != 1) return false;
    if (d->integrator != PHX_INT_RK4 && d->integrator != PHX_INT_DP54) return false;
    if ((size_t)d->nx * (size_t)d->ny > 0xffffffffull) return false;   // the noise counter holds the cell index in 32 bits
    return true;
}

Layout make_layout(const phx_grid_desc* d) {
    Layout L;
    std::memset(&L, 0, sizeof(L));
    const size_t rb = d->prec == PHX_C64 ? 8 : 4, cb = 2 * rb;
    const size_t plane = (size_t)d->nx * d->ny, cells = plane * d->batch;
    const int nc = model_spinor(d->model) ? 2 : 1;
    const bool res = model_reservoir(d->model);
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += align_up(bytes); return o; };
    for (int s = 0; s < nc; ++s) {
        L.psi[s] = take(cells * cb);
        L.ya[s] = take(cells * cb);
        L.yb[s] = take(cells * cb);
        L.acc[s] = take(cells * cb);
    }
    L.scratch_bytes = L.acc[0] + align_up(cells * cb) - L.yb[0];
    if (res)
        for (int s = 0; s < nc; ++s) {
            L.n[s] = take(cells * rb);
            L.na[s] = take(cells * rb);
            L.nb[s] = take(cells * rb);
            L.nacc[s] = take(cells * rb);
        }
    L.V = take(plane * rb);
    L.P = take(plane * rb);
    L.E = take(plane * cb);
    L.step = take(ALIGN);
    if (d->integrator == PHX_INT_DP54) {
        for (int q = 0; q < 7; ++q)
            for (int s = 0; s < nc; ++s) {
                L.K[q][s] = take(cells * cb);
                if (res) L.Kn[q][s] = take(cells * rb);
            }
        L.dpctl = take(sizeof(DpCtl));
        L.dplog = take((size_t)DP_LOG_CAP * (2 * sizeof(int) + 2 * sizeof(double)));
    }
    L.total = off;
    return L;
}

}  // namespace

struct phx_grid {
    phx_grid_desc d;
    Layout L;
    char* ws;
    cudaStream_t stream;
    cudaStream_t cap_stream;
    cudaStream_t side_stream;   // second branch of the captured step (the side launch of a ragged last strip)
    cudaEvent_t ev_fork, ev_join;
    int step_side;          // variant STEP side launch for a ragged last strip: 1 on; -1 and 0: off
    int step_pdl;           // variant STEP: later steps of a graph as programmatic dependent launches: -1 automatic, 0 off, 1 on
    int resident_cluster;   // variant RESIDENT cluster form: -1 automatic, 0 never, 1 whenever it applies
    bool has_params;
    phx_params prm;
    double coef[PHX_NCOEF];
    bool hasV, hasP, hasE;
    uint64_t step_host;
    uint64_t launches;
    int variant;            // resolved variant used by the next step
    int variant_req;        // requested (may be AUTO)
    int rows, vec, graph_steps, gsteps;
    int parity;             // variant STEP ping-pongs the state: 0 = state in psi/n, 1 = state in ya/na
    int step_ly, step_vec;  // variant STEP geometry (0 = automatic)
    int step_warps;         // variant STEP warps per CTA (0 = automatic)
    int step_bulk;          // variant STEP fetch path: -1 automatic, 0 register loads, 1 bulk copies into a shared-memory ring
    int step_xch;           // variant STEP exchanging strips (the warps of a CTA tile the whole row): -1 automatic, 0 off
    int async_host;         // 1: host copies of set_field / read_field do not synchronise (pinned buffers, caller syncs)
    cudaGraphExec_t g1[2], gN;  // one step from parity 0 / 1; graph_steps steps from parity 0
    cudaGraphExec_t gdp;        // adaptive integrator: setup -> WHILE { seven stages, control } -> finalize
    bool graphs_valid;
    int n_sm;
    size_t l2_bytes;        // L2 capacity of the device
    cudaError_t sticky;
    std::string err;
};

namespace {

phx_status fail(phx_grid* g, phx_status st, const char* msg) {
    if (g) g->err = msg;
    return st;
}

phx_status cuda_fail(phx_grid* g, cudaError_t e, const char* where) {
    if (g) {
        g->sticky = e;
        g->err = std::string(where) + ": " + cudaGetErrorString(e);
    }
    return PHX_ERR_CUDA;
}

#define PHX_CUDA(g, call)                                        \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return cuda_fail(g, e__, #call); \
    } while (0)

size_t real_bytes(const phx_grid* g) { return g->d.prec == PHX_C64 ? 8 : 4; }
size_t plane_cells(const phx_grid* g) { return (size_t)g->d.nx * g->d.ny; }

bool field_present(const phx_grid* g, int f) {
    const bool sp = model_spinor(g->d.model), rs = model_reservoir(g->d.model);
    switch (f) {
        case PHX_PSI: return true;
        case PHX_PSI_MINUS: return sp;
        case PHX_N: return rs;
        case PHX_N_MINUS: return rs && sp;
    }
    return false;
}

// Where the state field lives now (variant STEP alternates between the state buffer and the first stage buffer).
void* field_ptr(phx_grid* g, int f, size_t* bytes) {
    const size_t cells = plane_cells(g) * g->d.batch, rb = real_bytes(g);
    const bool alt = g->parity != 0;
    switch (f) {
        case PHX_PSI: *bytes = cells * 2 * rb; return g->ws + (alt ? g->L.ya[0] : g->L.psi[0]);
        case PHX_PSI_MINUS: *bytes = cells * 2 * rb; return g->ws + (alt ? g->L.ya[1] : g->L.psi[1]);
        case PHX_N: *bytes = cells * rb; return g->ws + (alt ? g->L.na[0] : g->L.n[0]);
        case PHX_N_MINUS: *bytes = cells * rb; return g->ws + (alt ? g->L.na[1] : g->L.n[1]);
    }
    *bytes = 0;
    return nullptr;
}

void drop_graphs(phx_grid* g) {
    for (int p = 0; p < 2; ++p) {
        if (g->g1[p]) cudaGraphExecDestroy(g->g1[p]);
        g->g1[p] = nullptr;
    }
    if (g->gN) cudaGraphExecDestroy(g->gN);
    g->gN = nullptr;
    if (g->gdp) cudaGraphExecDestroy(g->gdp);
    g->gdp = nullptr;
    g->graphs_valid = false;
}

template <typename T>
void fill_geo_coef(const phx_grid* g, Geom& geo, Coef<T>& k) {
    geo.nx = g->d.nx; geo.ny = g->d.ny; geo.batch = g->d.batch;
    geo.bc_x = g->d.bc_x; geo.bc_y = g->d.bc_y;
    geo.rows = g->rows;
    geo.pf = g->L.total > g->l2_bytes ? 1 : 0;      // (variant STAGE: L2 prefetch ahead of the register prefetch)
    geo.plane = plane_cells(g);
    const double* c = g->coef;
    k.cx = (T)c[0]; k.cy = (T)c[1]; k.ih = (T)c[2]; k.g = (T)c[3]; k.gx = (T)c[4]; k.gr = (T)c[5]; k.Rr = (T)c[6];
    k.hgc = (T)c[7]; k.gamr = (T)c[8]; k.bxx = (T)c[9]; k.byy = (T)c[10]; k.bxy = (T)c[11]; k.dt = (T)c[12];
    k.hdt = (T)(0.5 * c[12]);           // exact
    k.dt6 = (T)c[13]; k.dt3 = (T)c[14]; k.sig2 = (T)c[15]; k.doff = (T)c[16];
    const double r13 = c[13] / (0.5 * c[12]);
    k.r13 = (T)r13;
    k.r13lo = (T)(r13 - (double)k.r13);
    k.omega = c[17];
    k.dt_d = c[12];
}

template <typename T>
void fill_args(const phx_grid* g, StageArgs<T>& a) {
    using C = typename Cx<T>::type;
    std::memset(&a, 0, sizeof(a));
    fill_geo_coef<T>(g, a.geo, a.k);
    const int nc = model_spinor(g->d.model) ? 2 : 1;
    const bool res = model_reservoir(g->d.model);
    for (int s = 0; s < nc; ++s) {
        a.f.psi[s] = (C*)(g->ws + g->L.psi[s]);
        a.f.ya[s] = (C*)(g->ws + g->L.ya[s]);
        a.f.yb[s] = (C*)(g->ws + g->L.yb[s]);
        a.f.acc[s] = (C*)(g->ws + g->L.acc[s]);
        if (res) {
            a.f.n[s] = (T*)(g->ws + g->L.n[s]);
            a.f.na[s] = (T*)(g->ws + g->L.na[s]);
            a.f.nb[s] = (T*)(g->ws + g->L.nb[s]);
            a.f.nacc[s] = (T*)(g->ws + g->L.nacc[s]);
        }
    }
    a.f.V = g->hasV ? (const T*)(g->ws + g->L.V) : nullptr;
    a.f.P = g->hasP ? (const T*)(g->ws + g->L.P) : nullptr;
    a.f.E = g->hasE ? (const C*)(g->ws + g->L.E) : nullptr;
    a.f.step = (uint64_t*)(g->ws + g->L.step);
    a.seed = g->prm.seed;
}

// One RK4 step of variant STAGE: four fused stage kernels.
template <typename T>
cudaError_t enqueue_step_stage(phx_grid* g, cudaStream_t st) {
    StageArgs<T> a;
    fill_args<T>(g, a);
    const int vec = g->vec;
    const int tx = (g->d.nx + vec - 1) / vec;                   // threads needed along x
    int bx = ((tx + 31) / 32) * 32;
    if (bx > 128) bx = 128;
    const int by = 128 / bx;
    const dim3 block(bx, by, 1);
    const dim3 grid((tx + bx - 1) / bx, (g->d.ny + g->rows * by - 1) / (g->rows * by), g->d.batch);
    if (grid.y > 65535u) return cudaErrorInvalidConfiguration;
    for (int stage = 1; stage <= 4; ++stage) {
        cudaError_t e;
        const bool noise = g->d.noise != 0;
        if constexpr (sizeof(T) == 4) {
            switch (g->d.model) {
                case 0: e = launch_stage_32_0(a, stage, noise, vec, grid, block, st); break;
                case 1: e = launch_stage_32_1(a, stage, noise, vec, grid, block, st); break;
                case 2: e = launch_stage_32_2(a, stage, noise, vec, grid, block, st); break;
                default: e = launch_stage_32_3(a, stage, noise, vec, grid, block, st); break;
            }
        } else {
            switch (g->d.model) {
                case 0: e = launch_stage_64_0(a, stage, noise, vec, grid, block, st); break;
                case 1: e = launch_stage_64_1(a, stage, noise, vec, grid, block, st); break;
                case 2: e = launch_stage_64_2(a, stage, noise, vec, grid, block, st); break;
                default: e = launch_stage_64_3(a, stage, noise, vec, grid, block, st); break;
            }
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ---- variant STEP: launch plan ---------------------------------------------------------------------------------
int step_vec(const phx_grid* g) {
    if (g->step_vec) return g->step_vec;
    if (g->d.nx % 2 != 0) return 1;
    // complex fp64: two cells per lane (strips of 64 columns, 56 output columns instead of 24 of 32) on wide scalar grids
    if (g->d.prec != PHX_C32) return (g->d.model == PHX_SCALAR && g->d.nx >= 1024) ? 2 : 1;
    // four cells per lane: strips of 128 columns (120 output columns), 8 resident warps per SM; pays on wide scalar grids
    if (g->d.model == PHX_SCALAR && g->d.nx % 4 == 0 && g->d.nx >= 2048) return 4;
    return 2;
}

// dx == dy: the isotropic form of the Laplacian (cx == cy bit for bit, both derived from the same expression)
bool step_iso(const phx_grid* g) { return g->d.dx == g->d.dy; }

// Smallest workload (cells x realisations) AUTO gives the cp.async ring: same-run A/B, ring against register loads, Gcell*step/s:
// cfg3 physics 2048^2 144 / 124, 1024^2 94.7 / 90.5, 512^2 50.9 / 42.5; scalar fp32 1536^2 163.8 / 158.6, 1024^2 116.2 / 113.4,
// 512^2 59.8 / 50.9; scalar fp64 1024^2 73.0 / 71.7; below that the picture is mixed (384^2 fp32 29.9 / 31.8, 256^2 fp64
// 12.2 / 12.8, 256^2 fp32 19.4 / 18.3) and the register loads stay.
#ifndef PHX_RING_AUTO_LOG2_CELLS
#define PHX_RING_AUTO_LOG2_CELLS 18
#endif
// The bulk-copy fetch path (phx_step.cuh, BULK): periodic boundaries, rows whose pieces are 16-byte aligned and sized.
bool step_bulk(const phx_grid* g) {
    if (g->d.bc_x || g->d.bc_y) return false;
    if (((size_t)g->d.nx * real_bytes(g)) % 16 != 0) return false;
    if (g->d.nx < 32 * step_vec(g)) return false;       // a strip wraps at most once
    if (g->step_bulk >= 0) return g->step_bulk == 1;
    // automatic: the cp.async flavour of the ring where it measured faster than the register loads (phx_launch.h:
    // step_ring_auto), from 512^2 cells up, without drive; the TMA flavour stays an opt-in (slower everywhere)
    if (!step_ring_auto(g->d.prec == PHX_C64, g->d.model, step_vec(g)) || g->hasE) return false;
    return plane_cells(g) * g->d.batch >= ((size_t)1 << PHX_RING_AUTO_LOG2_CELLS);   // (small grids: the ring's prologue outweighs it)
}

int step_occupancy(const phx_grid* g, int vec) {
    const bool noise = g->d.noise != 0, zbc = g->d.bc_x || g->d.bc_y, iso = step_iso(g), drive = g->hasE, bulk = step_bulk(g);
    if (g->d.prec == PHX_C32) {
        switch (g->d.model) {
            case 0: return occupancy_step_32_0(noise, zbc, iso, drive, bulk, vec);
            case 1: return occupancy_step_32_1(noise, zbc, iso, drive, bulk, vec);
            case 2: return occupancy_step_32_2(noise, zbc, iso, drive, bulk, vec);
            default: return occupancy_step_32_3(noise, zbc, iso, drive, bulk, vec);
        }
    }
    switch (g->d.model) {
        case 0: return occupancy_step_64_0(noise, zbc, iso, drive, bulk, vec);
        case 1: return occupancy_step_64_1(noise, zbc, iso, drive, bulk, vec);
        case 2: return occupancy_step_64_2(noise, zbc, iso, drive, bulk, vec);
        default: return occupancy_step_64_3(noise, zbc, iso, drive, bulk, vec);
    }
}

// Ragged last strip.  The strips of 4 cells per lane produce 120 columns each: 4096 = 34 x 120 + 16, and a 35th strip (and
// with it 33 instead of 34 chunks of rows, to stay within one wave) would be computed for 16 columns.  When the remainder is at
// most a quarter of a strip, the main launch covers the whole strips only and a SIDE launch of the same kernel with one cell
// per lane (strips of 32 columns, a quarter of the work per row, 80 registers: its warps fit the register space the main launch
// leaves free) covers the remaining columns on a forked branch of the captured graph.  Only when asked for (tuning key
// step_side = 1): measured SLOWER, 179 against 204 Gcell*step/s at 4096^2 in the same run -- the two kernels of a step do not
// overlap (the side launch's 34 CTAs start when the main launch drains and then run alone for 11 us).
int stepx_vec(const phx_grid* g);
int step_side_cols(const phx_grid* g, int vec) {
    if (g->step_side != 1 || vec != 4 || stepx_vec(g) || step_bulk(g)) return 0;
    const int outw = 32 * vec - 8, rem = g->d.nx % outw;
    return (g->d.nx > outw && rem > 0 && rem <= outw / 4) ? rem : 0;
}

int step_strips(const phx_grid* g, int vec) {
    const int outw = 32 * vec - 8;
    return step_side_cols(g, vec) ? g->d.nx / outw : (g->d.nx + outw - 1) / outw;
}

// Warps per CTA: the warps of a CTA own adjacent strips and are otherwise independent.  Two per CTA measured 4 % faster
// than one on the 16384^2 spinor and equal on the 4096^2 reservoir grid; but a row with an odd number of strips leaves the
// last CTA's second warp idle: 1 of 6 warp slots on the 256-wide grids of cfg5 (5 strips: 91 against 75 Gcell*step/s with
// one warp per CTA), 1 of 36 at 4096^2 scalar fp32.  The launch plan (step_plan below) compares the two.
// Bytes one step of variant STEP touches per cell (state in and out, V, P, E).
size_t step_bytes_per_cell(const phx_grid* g) {
    const size_t rb = real_bytes(g);
    const size_t nc = model_spinor(g->d.model) ? 2 : 1;
    size_t b = nc * 4 * rb;
    if (model_reservoir(g->d.model)) b += nc * 2 * rb;
    if (g->hasV) b += rb;
    if (g->hasP) b += rb;
    if (g->hasE) b += 2 * rb;
    return b;
}

// Launch plan: rows per chunk (ly) and warps per CTA (wpc).  A chunk costs ly + 6 row iterations (4 + 4 halo rows and the
// pipeline fill, less the two rows the prologue fetches); the bulk-copy path runs whole passes of the unrolled row loop.
//  - Working set beyond L2 (the BASELINE grids from 4096^2 up, cfg5): an iteration waits on DRAM, more resident warps
//    hide it, and the grid runs in ceil(CTAs / resident CTAs) waves: minimise waves * iterations.
//  - Working set within half of L2 (1024^2): two warps per scheduler already saturate the FP32 pipe (measured at
//    1024^2 fp32: 525 cycles per iteration with 1-2 warps per scheduler, 810 with 3, 1250 with 4), so fewer, longer
//    chunks win: minimise iterations * max(1.75, warps per scheduler) (ly = 19 instead of 9: 113 instead of 80
//    Gcell*step/s).
//  One warp per CTA is taken when it is at least 2 % cheaper than two by this count (4096^2 scalar fp32: 35 strips x 33
//  chunks of 125 rows fill 1155 of 1184 warp slots, 131 iterations; in pairs 18 x 32 CTAs of 128 rows, 134 iterations).
struct StepPlan {
    int ly, wpc, vec;
    bool xch;
    int side_cols;      // > 0: the last side_cols columns of every row are left to a SIDE launch of one cell per lane
};

// Exchanging strips (phx_step.cuh, XCH): cells per lane with which the warps of one CTA tile the whole row, or 0.
// Periodic scalar / reservoir grids without drive whose width is 1 .. PHX_STEP_XWARPS strips of 32 * vec columns.
// Automatic (step_xch = -1): rows of at most 4 strips of 2 (fp64: 1) cells per lane on work of a million cells or more -- the
// ensembles of narrow grids, where the recomputed halo columns cost most (cfg5, 5 strips -> 4: 99.9 against 88.5
// Gcell*step/s; 512 x 64^2: 81.8 against 29.4).  A single small grid is latency-bound and the barrier per iteration costs it
// (64^2: 4.6 against 4.4 us per step), and 8 warps of 4 cells per lane on a 1024-wide row lose to the independent strips (80
// against 102-110): those run it only when asked for (step_xch = 1).
int stepx_vec(const phx_grid* g) {
    if (g->step_xch == 0) return 0;
    if (g->d.bc_x || g->d.bc_y || g->hasE || g->d.model > PHX_RESERVOIR) return 0;
    const bool forced = g->step_xch == 1;
    if (!forced && plane_cells(g) * g->d.batch < ((size_t)1 << 20)) return 0;
    for (int vec = 4; vec >= 1; vec >>= 1) {
        if (g->step_vec && vec != g->step_vec) continue;
        if (!stepx_has_vec(g->d.prec == PHX_C64, g->d.model, vec)) continue;
        const int w = 32 * vec;
        if (g->d.nx % w != 0 || g->d.nx / w > PHX_STEP_XWARPS) continue;
        if (!forced && (g->d.nx / w > 4 || vec > (g->d.prec == PHX_C64 ? 1 : 2))) continue;
        return vec;
    }
    return 0;
}

int stepx_occupancy(const phx_grid* g, int vec, int warps) {
    const bool noise = g->d.noise != 0, iso = step_iso(g);
    if (g->d.prec == PHX_C32)
        return g->d.model == 0 ? occupancy_stepx_32_0(noise, iso, vec, warps) : occupancy_stepx_32_1(noise, iso, vec, warps);
    return g->d.model == 0 ? occupancy_stepx_64_0(noise, iso, vec, warps) : occupancy_stepx_64_1(noise, iso, vec, warps);
}

double step_plan_cost(const phx_grid* g, int vec, int wpc, int* ly_out, bool xch = false) {
    const int strips = xch ? wpc : step_strips(g, vec);
    const long ctas_row = (long)((strips + wpc - 1) / wpc) * g->d.batch;
    const long slots = xch ? (long)g->n_sm * stepx_occupancy(g, vec, wpc)
                           : (long)g->n_sm * step_occupancy(g, vec) * (PHX_STEP_WARPS / wpc);   // resident CTAs of wpc warps
    const bool in_l2 = plane_cells(g) * g->d.batch * step_bytes_per_cell(g) < g->l2_bytes / 2;
    const bool whole_passes = xch || (step_bulk(g) && !step_ring_cpasync(g->d.prec == PHX_C64, g->d.model, vec)) ||
                              !step_early_exit(g->d.prec == PHX_C64, g->d.model, vec);
    const int ring = xch ? 4 + step_xch_lead(g->d.prec == PHX_C64, g->d.model, vec) : PHX_STEP_RING;
    double best_cost = -1;
    int best_ly = g->d.ny;
    const int max_chunks = g->d.ny / 4 > 0 ? g->d.ny / 4 : 1;   // (a 64^2 grid: ly = 4, 3.6 instead of 4.9 us per step)
    for (int nch = 1; nch <= max_chunks && nch <= 65535; ++nch) {
        int ly = (g->d.ny + nch - 1) / nch;
        if (g->step_ly) ly = g->step_ly < g->d.ny ? g->step_ly : g->d.ny;
        const int real_chunks = (g->d.ny + ly - 1) / ly;
        const long ctas = ctas_row * real_chunks;
        const long waves = (ctas + slots - 1) / slots;
        const long iters = whole_passes ? (ly + 6 + ring - 1) / ring * ring : ly + 6;
        double cost = (double)(waves * iters);
        if (in_l2) {
            const long per_sm = ((ctas + waves - 1) / waves + g->n_sm - 1) / g->n_sm;     // CTAs on the fullest SM
            const long per_sched = (per_sm * wpc + 3) / 4;
            cost *= per_sched > 1.75 ? (double)per_sched : 1.75;
        }
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_ly = ly; }
        if (g->step_ly) break;
    }
    // Chunks that start on a multiple of 64 rows when that costs at most 2.5 % more by the count above (4096^2 fp32, same
    // run: ly = 128 216.2, ly = 125 213.1 Gcell*step/s although 125 rows are 131 iterations against 134: the rows of a chunk
    // boundary then start on the same DRAM page stride for every warp).
    if (!g->step_ly && !in_l2 && best_ly % 64 != 0) {
        const int ly = (best_ly + 63) / 64 * 64;
        if (ly < g->d.ny) {
            const long ctas = ctas_row * ((g->d.ny + ly - 1) / ly);
            const long waves = (ctas + slots - 1) / slots;
            const long iters = whole_passes ? (ly + 6 + ring - 1) / ring * ring : ly + 6;
            const double cost = (double)(waves * iters);
            if (cost <= best_cost * 1.025) { best_cost = cost; best_ly = ly; }
        }
    }
    *ly_out = best_ly;
    return best_cost;
}

StepPlan step_plan(const phx_grid* g) {
    StepPlan p;
    p.xch = false;
    p.side_cols = 0;
    if (const int xv = stepx_vec(g)) {
        p.xch = true;
        p.vec = xv;
        p.wpc = g->d.nx / (32 * xv);
        step_plan_cost(g, xv, p.wpc, &p.ly, true);
        return p;
    }
    const int vec = p.vec = step_vec(g);
    p.side_cols = step_side_cols(g, vec);
    if (g->step_warps) {
        p.wpc = g->step_warps;
        step_plan_cost(g, vec, p.wpc, &p.ly);
        return p;
    }
    int ly2 = 0, ly1 = 0;
    const double c2 = step_plan_cost(g, vec, PHX_STEP_WARPS, &ly2), c1 = step_plan_cost(g, vec, 1, &ly1);
    const int strips = step_strips(g, vec);
    const bool idle_warp = strips % PHX_STEP_WARPS != 0 && strips < 50;   // pairs would leave more than 2 % of the warp slots idle
    if (c1 * 1.02 < c2 || (idle_warp && c1 <= c2 * 1.02)) { p.wpc = 1; p.ly = ly1; }
    else { p.wpc = PHX_STEP_WARPS; p.ly = ly2; }
    return p;
}

// One RK4 step of variant STEP: a single kernel that reads the state of parity p and writes parity 1-p.
// pdl: launch as a programmatic dependent of the previous kernel in the stream (the later steps of a captured graph)
template <typename T>
cudaError_t enqueue_step_fused(phx_grid* g, cudaStream_t st, int parity, bool pdl = false) {
    using C = typename Cx<T>::type;
    StepArgs<T> a;
    std::memset(&a, 0, sizeof(a));
    fill_geo_coef<T>(g, a.geo, a.k);
    const int nc = model_spinor(g->d.model) ? 2 : 1;
    const bool res = model_reservoir(g->d.model);
    for (int s = 0; s < nc; ++s) {
        C* main_ = (C*)(g->ws + g->L.psi[s]);
        C* alt = (C*)(g->ws + g->L.ya[s]);
        a.psi_in[s] = parity ? alt : main_;
        a.psi_out[s] = parity ? main_ : alt;
        if (res) {
            T* nmain = (T*)(g->ws + g->L.n[s]);
            T* nalt = (T*)(g->ws + g->L.na[s]);
            a.n_in[s] = parity ? nalt : nmain;
            a.n_out[s] = parity ? nmain : nalt;
        }
    }
    a.V = g->hasV ? (const T*)(g->ws + g->L.V) : nullptr;
    a.P = g->hasP ? (const T*)(g->ws + g->L.P) : nullptr;
    a.E = g->hasE ? (const C*)(g->ws + g->L.E) : nullptr;
    uint64_t* slots = (uint64_t*)(g->ws + g->L.step);
    a.step_in = slots + parity;
    a.step_out = slots + (1 - parity);
    a.seed = g->prm.seed;
    a.pdl = pdl ? 1 : 0;
    const StepPlan plan = step_plan(g);
    const int vec = plan.vec;
    a.strips = plan.xch ? plan.wpc : step_strips(g, vec);
    a.wpc = plan.wpc;
    a.ly = plan.ly;
    const dim3 grid((a.strips + a.wpc - 1) / a.wpc, (g->d.ny + a.ly - 1) / a.ly, g->d.batch);
    if (grid.y > 65535u) return cudaErrorInvalidConfiguration;
    const bool noise = g->d.noise != 0, zbc = g->d.bc_x || g->d.bc_y, iso = step_iso(g), bulk = step_bulk(g);
    if (plan.xch) {
        if constexpr (sizeof(T) == 4)
            return g->d.model == 0 ? launch_stepx_32_0(a, noise, iso, vec, grid, st) : launch_stepx_32_1(a, noise, iso, vec, grid, st);
        else
            return g->d.model == 0 ? launch_stepx_64_0(a, noise, iso, vec, grid, st) : launch_stepx_64_1(a, noise, iso, vec, grid, st);
    }
    auto launch = [&](const StepArgs<T>& args, int v, dim3 gr, cudaStream_t stream) -> cudaError_t {
        if constexpr (sizeof(T) == 4) {
            switch (g->d.model) {
                case 0: return launch_step_32_0(args, noise, zbc, iso, bulk, v, gr, stream);
                case 1: return launch_step_32_1(args, noise, zbc, iso, bulk, v, gr, stream);
                case 2: return launch_step_32_2(args, noise, zbc, iso, bulk, v, gr, stream);
                default: return launch_step_32_3(args, noise, zbc, iso, bulk, v, gr, stream);
            }
        } else {
            switch (g->d.model) {
                case 0: return launch_step_64_0(args, noise, zbc, iso, bulk, v, gr, stream);
                case 1: return launch_step_64_1(args, noise, zbc, iso, bulk, v, gr, stream);
                case 2: return launch_step_64_2(args, noise, zbc, iso, bulk, v, gr, stream);
                default: return launch_step_64_3(args, noise, zbc, iso, bulk, v, gr, stream);
            }
        }
    };
    if (plan.side_cols == 0) return launch(a, vec, grid, st);
    // main launch (whole strips) and side launch (the remaining columns, one cell per lane) on two branches
    a.pdl = 0;      // (events between the branches: ordinary dependencies)
    cudaError_t e = cudaEventRecord(g->ev_fork, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(g->side_stream, g->ev_fork, 0);
    if (e == cudaSuccess) e = launch(a, vec, grid, st);
    if (e != cudaSuccess) return e;
    StepArgs<T> b = a;
    b.x0 = a.strips * (32 * vec - 8);
    b.strips = (plan.side_cols + 23) / 24;
    b.wpc = 1;
    e = launch(b, 1, dim3(b.strips, grid.y, grid.z), g->side_stream);
    if (e == cudaSuccess) e = cudaEventRecord(g->ev_join, g->side_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, g->ev_join, 0);
    return e;
}

// Programmatic dependent launches inside a graph of fused steps (the CTAs of step s+1 are scheduled early and wait in
// griddepcontrol.wait for step s): hides the launch latency, which is all a tiny grid has -- one 64^2 grid 3.33 against 3.58 us
// per step, cfg1 3.59 against 3.84, 256^2 3.59 against 3.84 -- but CTAs that are placed while the previous grid still holds
// most SMs end up unevenly spread: 512^2 -5 %, 1024^2 82 against 113 Gcell*step/s, 4096^2 -3 %.  Automatic: up to 256^2 cells.
bool step_pdl_wanted(const phx_grid* g) {
    if (g->step_pdl == 0 || g->variant != PHX_VARIANT_STEP) return false;
    if (g->step_pdl == 1) return true;
    return plane_cells(g) * g->d.batch <= (size_t)256 * 256;
}

int kernels_per_step(const phx_grid* g) {
    if (g->variant != PHX_VARIANT_STEP) return 4;
    return step_plan(g).side_cols > 0 ? 2 : 1;      // (a ragged last strip: main + side launch)
}   // (RESIDENT: one per call)

// Variant RESIDENT, which form: the cluster form (one realisation on 2-8 CTAs) when the grid does not fit one CTA, and for
// small batches -- one 64^2 grid is stepped 2x faster by 8 SMs with a cluster barrier per stage than by one SM -- unless
// the tuning key resident_cluster says otherwise (0 never, 1 whenever it applies).
bool resident_single_ok(const phx_grid* g) {
    return resident_cpt(plane_cells(g), g->d.prec == PHX_C64, model_reservoir(g->d.model)) != 0;
}
int resident_cluster_ctas(const phx_grid* g) {
    return resident_cluster_size(g->d.nx, g->d.ny, g->d.prec == PHX_C64, model_reservoir(g->d.model));
}
bool resident_use_cluster(const phx_grid* g) {
    const int n = resident_cluster_ctas(g);
    if (n == 0 || g->resident_cluster == 0) return false;
    if (g->hasE) return true;                                 // (a drive: only the cluster form of the scalar model carries it)
    if (!resident_single_ok(g) || g->resident_cluster == 1) return true;
    return (long)g->d.batch * n <= (long)g->n_sm;          // every cluster resident at once: more SMs per realisation
}

// Variant RESIDENT: all n steps in one launch, in place on the buffers of the current parity.
template <typename T>
cudaError_t launch_resident(phx_grid* g, int n_steps) {
    using C = typename Cx<T>::type;
    ResidentArgs<T> a;
    std::memset(&a, 0, sizeof(a));
    fill_geo_coef<T>(g, a.geo, a.k);
    const bool res = model_reservoir(g->d.model);
    a.psi = (C*)(g->ws + (g->parity ? g->L.ya[0] : g->L.psi[0]));
    a.n = res ? (T*)(g->ws + (g->parity ? g->L.na[0] : g->L.n[0])) : nullptr;
    a.V = g->hasV ? (const T*)(g->ws + g->L.V) : nullptr;
    a.P = g->hasP ? (const T*)(g->ws + g->L.P) : nullptr;
    a.E = g->hasE ? (const C*)(g->ws + g->L.E) : nullptr;
    a.step_slots = (uint64_t*)(g->ws + g->L.step);
    a.step0 = g->step_host;
    a.n_steps = n_steps;
    a.seed = g->prm.seed;
    if (resident_use_cluster(g)) {
        if constexpr (sizeof(T) == 4) return launch_resident_cluster_32(a, res, g->d.noise != 0, g->stream);
        else return launch_resident_cluster_64(a, res, g->d.noise != 0, g->stream);
    }
    if constexpr (sizeof(T) == 4) return launch_resident_32(a, res, g->d.noise != 0, g->stream);
    else return launch_resident_64(a, res, g->d.noise != 0, g->stream);
}

// Enqueues one step starting from state parity `parity` (always 0 for variant STAGE).
cudaError_t enqueue_step(phx_grid* g, cudaStream_t st, int parity, bool pdl = false) {
    if (g->variant == PHX_VARIANT_STEP)
        return g->d.prec == PHX_C64 ? enqueue_step_fused<double>(g, st, parity, pdl) : enqueue_step_fused<float>(g, st, parity, pdl);
    return g->d.prec == PHX_C64 ? enqueue_step_stage<double>(g, st) : enqueue_step_stage<float>(g, st);
}

cudaError_t capture(phx_grid* g, int steps, int parity, cudaGraphExec_t* out) {
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(g->cap_stream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return e;
    cudaError_t le = cudaSuccess;
    for (int s = 0; s < steps && le == cudaSuccess; ++s) {
        le = enqueue_step(g, g->cap_stream, parity, s > 0 && step_pdl_wanted(g));
        if (g->variant == PHX_VARIANT_STEP) parity ^= 1;
    }
    e = cudaStreamEndCapture(g->cap_stream, &graph);
    if (le != cudaSuccess) { if (graph) cudaGraphDestroy(graph); return le; }
    if (e != cudaSuccess) return e;
    e = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    return e;
}

// The fused step addresses a plane by 32-bit cell offsets.
bool step_variant_ok(const phx_grid* g) { return (size_t)g->d.nx * (size_t)g->d.ny < ((size_t)1 << 31); }

// Variant RESIDENT: scalar and reservoir models without drive whose grid fits one CTA (phx_resident.cu).
bool resident_variant_ok(const phx_grid* g) {
    if (model_spinor(g->d.model)) return false;
    if (g->hasE) return g->d.model == PHX_SCALAR && g->resident_cluster != 0 && resident_drive_ok(g->d.nx, g->d.ny, g->d.prec == PHX_C64);
    return resident_single_ok(g) || (g->resident_cluster != 0 && resident_cluster_ctas(g) != 0);
}

// Largest single grid AUTO gives to the cluster form of variant RESIDENT (measured, us per step, clusters of 16 CTAs against the
// fused step: cfg1 64^2 fp64 2.23 / 3.58, 64^2 fp32 1.74 / 3.33, 128^2 fp32 2.92 / 3.38, 128^2 fp64 3.53 / 3.92).
constexpr int RESIDENT_CLUSTER_AUTO_CELLS = 16384;

// AUTO takes the resident kernel for ensembles of grids that fit it (one CTA per realisation: 2.3x the fused step on
// 512 x 64^2 fp32; a single small grid is faster spread over several SMs by the fused step: 3.9 against 4.3 us per step at
// 64^2 fp32), else the fused step wherever it can run (1.4-4.7x faster than the per-stage kernels on every BASELINE
// workload); STAGE runs every model, size and term.
void resolve_variant(phx_grid* g) {
    const int req = g->variant_req;
    const bool res_ok = resident_variant_ok(g);
    // (AUTO: ensembles of grids that fit one CTA; single grids of at most 128^2 cells on a cluster)
    const bool auto_res = g->d.batch >= 32 ? resident_single_ok(g)
                                           : (resident_use_cluster(g) && plane_cells(g) <= (size_t)RESIDENT_CLUSTER_AUTO_CELLS);
    if (res_ok && (req == PHX_VARIANT_RESIDENT || (req == PHX_VARIANT_AUTO && auto_res))) g->variant = PHX_VARIANT_RESIDENT;
    else if (req != PHX_VARIANT_STAGE && step_variant_ok(g)) g->variant = PHX_VARIANT_STEP;
    else g->variant = PHX_VARIANT_STAGE;
}

// Variant STAGE keeps the state in psi/n: if the fused-step ping-pong left it in the alternate buffers, move it
// back (and realign the device step-counter slots) before another variant runs.
phx_status normalise_state(phx_grid* g) {
    if (g->parity == 0) return PHX_OK;
    const int nc = model_spinor(g->d.model) ? 2 : 1;
    const size_t cells = plane_cells(g) * g->d.batch, rb = real_bytes(g);
    for (int s = 0; s < nc; ++s) {
        PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.psi[s], g->ws + g->L.ya[s], cells * 2 * rb, cudaMemcpyDeviceToDevice, g->stream));
        if (model_reservoir(g->d.model))
            PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.n[s], g->ws + g->L.na[s], cells * rb, cudaMemcpyDeviceToDevice, g->stream));
    }
    const uint64_t slots[2] = {g->step_host, g->step_host};
    PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.step, slots, sizeof(slots), cudaMemcpyHostToDevice, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    g->parity = 0;
    return PHX_OK;
}

// Re-resolves the variant after a request or a change of the terms present; drops the captured graphs.
phx_status apply_variant(phx_grid* g) {
    resolve_variant(g);
    drop_graphs(g);
    if (g->variant == PHX_VARIANT_STAGE) return normalise_state(g);   // STAGE keeps the state in psi/n
    return PHX_OK;
}

phx_status copy_in(phx_grid* g, void* dst, const void* src, size_t bytes, phx_mem where) {
    if (where == PHX_HOST) {
        PHX_CUDA(g, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, g->stream));
        if (!g->async_host) PHX_CUDA(g, cudaStreamSynchronize(g->stream));   // the caller may reuse a pageable source at once
    } else {
        PHX_CUDA(g, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, g->stream));
    }
    return PHX_OK;
}

phx_status copy_out(phx_grid* g, void* dst, const void* src, size_t bytes, phx_mem where) {
    PHX_CUDA(g, cudaMemcpyAsync(dst, src, bytes, where == PHX_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice,
                                g->stream));
    if (!(g->async_host && where == PHX_HOST)) PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    return PHX_OK;
}

// ---- adaptive Dormand-Prince 5(4) (phx_adaptive.cu) --------------------------------------------------------------------------
DpCtl* dp_ctl(phx_grid* g) { return (DpCtl*)(g->ws + g->L.dpctl); }

template <typename T>
void fill_dp_args(phx_grid* g, DpArgs<T>& a) {
    using C = typename Cx<T>::type;
    std::memset(&a, 0, sizeof(a));
    fill_geo_coef<T>(g, a.geo, a.k);
    const int nc = model_spinor(g->d.model) ? 2 : 1;
    const bool res = model_reservoir(g->d.model);
    for (int s = 0; s < nc; ++s) {
        a.S[0][s] = (C*)(g->ws + g->L.psi[s]);
        a.S[1][s] = (C*)(g->ws + g->L.acc[s]);
        a.Y[0][s] = (C*)(g->ws + g->L.ya[s]);
        a.Y[1][s] = (C*)(g->ws + g->L.yb[s]);
        for (int q = 0; q < 7; ++q) a.K[q][s] = (C*)(g->ws + g->L.K[q][s]);
        if (res) {
            a.Sn[0][s] = (T*)(g->ws + g->L.n[s]);
            a.Sn[1][s] = (T*)(g->ws + g->L.nacc[s]);
            a.Yn[0][s] = (T*)(g->ws + g->L.na[s]);
            a.Yn[1][s] = (T*)(g->ws + g->L.nb[s]);
            for (int q = 0; q < 7; ++q) a.Kn[q][s] = (T*)(g->ws + g->L.Kn[q][s]);
        }
    }
    a.V = g->hasV ? (const T*)(g->ws + g->L.V) : nullptr;
    a.P = g->hasP ? (const T*)(g->ws + g->L.P) : nullptr;
    a.E = g->hasE ? (const C*)(g->ws + g->L.E) : nullptr;
    a.ctl = dp_ctl(g);
    // Dormand & Prince, J. Comput. Appl. Math. 6 (1980) 19: each coefficient a double quotient, rounded once to T
    const double A[7][7] = {
        {0, 0, 0, 0, 0, 0, 0},
        {1.0 / 5.0, 0, 0, 0, 0, 0, 0},
        {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0, 0},
        {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0, 0},
        {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0, 0},
        {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0, 0},
        {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0}};
    const double BS[7] = {5179.0 / 57600.0, 0.0, 7571.0 / 16695.0, 393.0 / 640.0, -92097.0 / 339200.0, 187.0 / 2100.0, 1.0 / 40.0};
    const double Cn[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
    for (int s = 0; s < 7; ++s) {
        a.c[s] = (T)Cn[s];
        a.e[s] = (T)(A[6][s] - BS[s]);
        for (int q = 0; q < 7; ++q) a.a[s][q] = (T)A[s][q];
    }
}

// Builds the graph  setup -> WHILE { stage 1..7, control } -> finalize  once per handle (it depends on pointers and geometry
// only; tolerances and t_end travel through the device control block).
template <typename T>
cudaError_t build_dp_graph(phx_grid* g) {
    DpArgs<T> a;
    fill_dp_args<T>(g, a);
    const int prec32 = g->d.prec == PHX_C32;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaGraphCreate(&graph, 0);
    if (e != cudaSuccess) return e;
    auto bail = [&](cudaError_t err) { cudaGraphDestroy(graph); return err; };
    cudaGraphConditionalHandle handle;
    e = cudaGraphConditionalHandleCreate(&handle, graph, 0, 0);
    if (e != cudaSuccess) return bail(e);
    // (1) setup kernel
    e = cudaStreamBeginCaptureToGraph(g->cap_stream, graph, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return bail(e);
    cudaError_t le = dp_launch_setup(a.ctl, (unsigned long long)handle, prec32, g->cap_stream);
    e = cudaStreamEndCapture(g->cap_stream, &graph);
    if (le != cudaSuccess) return bail(le);
    if (e != cudaSuccess) return bail(e);
    cudaGraphNode_t setup_node = nullptr;
    size_t nn = 1;
    e = cudaGraphGetNodes(graph, &setup_node, &nn);
    if (e != cudaSuccess || nn != 1) return bail(e != cudaSuccess ? e : cudaErrorUnknown);
    // (2) the WHILE node
    cudaGraphNodeParams cp = {cudaGraphNodeTypeConditional};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = handle;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    cudaGraphNode_t while_node = nullptr;
    e = cudaGraphAddNode(&while_node, graph, &setup_node, 1, &cp);
    if (e != cudaSuccess) return bail(e);
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    e = cudaStreamBeginCaptureToGraph(g->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return bail(e);
    le = dp_launch_attempt<T>(a, g->d.model, g->cap_stream);
    if (le == cudaSuccess) le = dp_launch_control(a.ctl, (unsigned long long)handle, prec32, DP_LOG_CAP, g->cap_stream);
    e = cudaStreamEndCapture(g->cap_stream, &body);
    if (le != cudaSuccess) return bail(le);
    if (e != cudaSuccess) return bail(e);
    // (3) finalize, after the loop
    e = cudaStreamBeginCaptureToGraph(g->cap_stream, graph, &while_node, nullptr, 1, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return bail(e);
    le = dp_launch_finalize<T>(a, g->d.model, g->n_sm, g->cap_stream);
    e = cudaStreamEndCapture(g->cap_stream, &graph);
    if (le != cudaSuccess) return bail(le);
    if (e != cudaSuccess) return bail(e);
    e = cudaGraphInstantiate(&g->gdp, graph, 0);
    cudaGraphDestroy(graph);
    return e;
}

}  // namespace

extern "C" {

size_t phx_workspace_bytes(const phx_grid_desc* desc) {
    if (!desc_ok(desc)) return 0;
    return make_layout(desc).total;
}

phx_status phx_create_grid(phx_grid** out, const phx_grid_desc* desc) {
    if (!out) return PHX_ERR_INVALID_ARG;
    *out = nullptr;
    if (!desc_ok(desc)) return PHX_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return PHX_ERR_CUDA;   // no CPU fallback
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return PHX_ERR_CUDA;
    if (prop.major != 10) return PHX_ERR_CUDA;   // the kernels are built for sm_100a only
    const Layout L = make_layout(desc);
    if (!desc->workspace || ((uintptr_t)desc->workspace % ALIGN) != 0 || desc->workspace_bytes < L.total)
        return PHX_ERR_WORKSPACE;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, desc->workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return PHX_ERR_WORKSPACE;
    }
    phx_grid* g = new (std::nothrow) phx_grid();
    if (!g) return PHX_ERR_INVALID_ARG;
    g->d = *desc;
    g->L = L;
    g->ws = (char*)desc->workspace;
    g->stream = (cudaStream_t)desc->stream;
    g->cap_stream = nullptr;
    g->side_stream = nullptr;
    g->ev_fork = nullptr;
    g->ev_join = nullptr;
    g->has_params = false;
    std::memset(&g->prm, 0, sizeof(g->prm));
    std::memset(g->coef, 0, sizeof(g->coef));
    g->hasV = g->hasP = g->hasE = false;
    g->step_host = 0;
    g->launches = 0;
    g->variant_req = PHX_VARIANT_AUTO;
    g->rows = 16;
    g->vec = (desc->prec == PHX_C32 && desc->nx % 2 == 0) ? 2 : 1;
    g->graph_steps = g->gsteps = 8;
    g->g1[0] = g->g1[1] = g->gN = nullptr;
    g->gdp = nullptr;
    g->graphs_valid = false;
    g->parity = 0;
    g->step_ly = g->step_vec = 0;
    g->step_bulk = -1;
    g->step_xch = -1;
    g->step_side = -1;
    g->step_pdl = -1;
    g->resident_cluster = -1;
    g->step_warps = 0;
    g->async_host = 0;
    g->n_sm = prop.multiProcessorCount;
    g->l2_bytes = (size_t)prop.l2CacheSize;
    g->sticky = cudaSuccess;
    g->variant = PHX_VARIANT_STAGE;
    resolve_variant(g);
    if (cudaStreamCreateWithFlags(&g->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { delete g; return PHX_ERR_CUDA; }
    if (cudaStreamCreateWithFlags(&g->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&g->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&g->ev_join, cudaEventDisableTiming) != cudaSuccess) { delete g; return PHX_ERR_CUDA; }
    // zero the state, the static fields and the step counter
    if (cudaMemsetAsync(g->ws, 0, L.total, g->stream) != cudaSuccess) { cudaStreamDestroy(g->cap_stream); delete g; return PHX_ERR_CUDA; }
    if (desc->integrator == PHX_INT_DP54) {
        // the control block is all zeros (t = 0, no proposal pending); its log arrays follow it in the workspace
        DpCtl c;
        std::memset(&c, 0, sizeof(c));
        char* lg = g->ws + L.dplog;
        c.log_accept = (int*)lg;
        c.log_q = (int*)(lg + (size_t)DP_LOG_CAP * sizeof(int));
        c.log_h = (double*)(lg + (size_t)DP_LOG_CAP * 2 * sizeof(int));
        c.log_err = (double*)(lg + (size_t)DP_LOG_CAP * (2 * sizeof(int) + sizeof(double)));
        if (cudaMemcpyAsync(g->ws + L.dpctl, &c, sizeof(c), cudaMemcpyHostToDevice, g->stream) != cudaSuccess ||
            cudaStreamSynchronize(g->stream) != cudaSuccess) {
            cudaStreamDestroy(g->cap_stream);
            delete g;
            return PHX_ERR_CUDA;
        }
    }
    *out = g;
    return PHX_OK;
}

phx_status phx_set_params(phx_grid* g, const phx_params* p) {
    if (!g || !p) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!(p->dt > 0) || p->hbar == 0 || p->m == 0 || !std::isfinite(p->hbar) || !std::isfinite(p->m) || !std::isfinite(p->dt))
        return fail(g, PHX_ERR_INVALID_ARG, "phx_set_params: dt must be > 0 and hbar, m non-zero");
    const double dx = g->d.dx, dy = g->d.dy;
    double c[PHX_NCOEF];
    // canonical coefficient set (step 0): double expressions, each rounded once to T
    c[0] = p->hbar / (2.0 * p->m * dx * dx);
    c[1] = p->hbar / (2.0 * p->m * dy * dy);
    c[2] = 1.0 / p->hbar;
    c[3] = p->g;
    c[4] = p->g_x;
    c[5] = p->g_r;
    c[6] = p->R;
    c[7] = p->gamma_c / 2.0;
    c[8] = p->gamma_r;
    c[9] = p->beta / (p->hbar * dx * dx);
    c[10] = p->beta / (p->hbar * dy * dy);
    c[11] = p->beta / (2.0 * p->hbar * dx * dy);
    c[12] = p->dt;
    c[13] = p->dt / 6.0;
    c[14] = p->dt / 3.0;
    c[15] = p->noise_scale * p->dt / (4.0 * dx * dy);
    c[16] = p->density_offset;
    c[17] = p->omega;
    for (int i = 0; i < PHX_NCOEF; ++i) {
        if (!std::isfinite(c[i])) return fail(g, PHX_ERR_INVALID_ARG, "phx_set_params: non-finite coefficient");
        g->coef[i] = g->d.prec == PHX_C32 ? (double)(float)c[i] : c[i];
    }
    g->prm = *p;
    g->has_params = true;
    drop_graphs(g);
    const double wmax = std::fabs(p->hbar / (2.0 * p->m)) * (4.0 / (dx * dx) + 4.0 / (dy * dy)) * p->dt;
    if (wmax > 2.78) {
        g->err = "phx_set_params: (hbar/2m)(4/dx^2+4/dy^2) dt exceeds the RK4 stability limit 2.78";
        return PHX_WARN_UNSTABLE;
    }
    return PHX_OK;
}

phx_status phx_set_potential_pump(phx_grid* g, const void* V, const void* P, phx_mem where) {
    if (!g || (where != PHX_HOST && where != PHX_DEVICE)) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (P && !model_reservoir(g->d.model))
        return fail(g, PHX_ERR_UNSUPPORTED, "phx_set_potential_pump: a pump P needs a model with a reservoir (Eq. (17))");
    const size_t bytes = plane_cells(g) * real_bytes(g);
    if (V) { phx_status s = copy_in(g, g->ws + g->L.V, V, bytes, where); if (s) return s; }
    if (P) { phx_status s = copy_in(g, g->ws + g->L.P, P, bytes, where); if (s) return s; }
    if (g->hasV != (V != nullptr) || g->hasP != (P != nullptr)) drop_graphs(g);
    g->hasV = V != nullptr;
    g->hasP = P != nullptr;
    return PHX_OK;
}

phx_status phx_set_drive(phx_grid* g, const void* E, phx_mem where) {
    if (!g || (where != PHX_HOST && where != PHX_DEVICE)) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (E) { phx_status s = copy_in(g, g->ws + g->L.E, E, plane_cells(g) * 2 * real_bytes(g), where); if (s) return s; }
    const bool changed = g->hasE != (E != nullptr);
    g->hasE = E != nullptr;
    if (changed) return apply_variant(g);
    return PHX_OK;
}

phx_status phx_set_field(phx_grid* g, phx_field f, const void* src, phx_mem where) {
    if (!g || !src || (where != PHX_HOST && where != PHX_DEVICE) || f < PHX_PSI || f > PHX_N_MINUS) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!field_present(g, f)) return fail(g, PHX_ERR_UNSUPPORTED, "phx_set_field: field not present in this model");
    size_t bytes;
    void* dst = field_ptr(g, f, &bytes);
    return copy_in(g, dst, src, bytes, where);
}

phx_status phx_read_field(phx_grid* g, phx_field f, void* dst, phx_mem where) {
    if (!g || !dst || (where != PHX_HOST && where != PHX_DEVICE) || f < PHX_PSI || f > PHX_N_MINUS) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!field_present(g, f)) return fail(g, PHX_ERR_UNSUPPORTED, "phx_read_field: field not present in this model");
    size_t bytes;
    void* src = field_ptr(g, f, &bytes);
    return copy_out(g, dst, src, bytes, where);
}

phx_status phx_step_rk4(phx_grid* g, int64_t n_steps) {
    if (!g || n_steps < 0) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!g->has_params) return fail(g, PHX_ERR_BAD_STATE, "phx_step_rk4: call phx_set_params first");
    if (n_steps == 0) return PHX_OK;
    if (g->variant == PHX_VARIANT_RESIDENT) {
        for (int64_t left = n_steps; left > 0;) {
            const int chunk = left > (1 << 30) ? (1 << 30) : (int)left;
            PHX_CUDA(g, g->d.prec == PHX_C64 ? launch_resident<double>(g, chunk) : launch_resident<float>(g, chunk));
            g->step_host += (uint64_t)chunk;
            g->launches += 1;
            left -= chunk;
        }
        return PHX_OK;
    }
    if (!g->graphs_valid) {
        drop_graphs(g);
        PHX_CUDA(g, capture(g, 1, 0, &g->g1[0]));
        if (g->variant == PHX_VARIANT_STEP) PHX_CUDA(g, capture(g, 1, 1, &g->g1[1]));
        // the multi-step graph of the ping-pong variant must return to parity 0: an even number of steps
        g->gsteps = g->variant == PHX_VARIANT_STEP ? (g->graph_steps < 2 ? 2 : g->graph_steps & ~1) : g->graph_steps;
        PHX_CUDA(g, capture(g, g->gsteps, 0, &g->gN));
        g->graphs_valid = true;
    }
    const bool pingpong = g->variant == PHX_VARIANT_STEP;
    int64_t left = n_steps;
    if (pingpong && g->parity == 1) {   // the multi-step graph is captured from parity 0
        PHX_CUDA(g, cudaGraphLaunch(g->g1[1], g->stream));
        g->parity = 0;
        --left;
    }
    while (left >= g->gsteps) {
        PHX_CUDA(g, cudaGraphLaunch(g->gN, g->stream));
        left -= g->gsteps;
    }
    while (left > 0) {
        PHX_CUDA(g, cudaGraphLaunch(g->g1[pingpong ? g->parity : 0], g->stream));
        if (pingpong) g->parity ^= 1;
        --left;
    }
    g->step_host += (uint64_t)n_steps;
    g->launches += (uint64_t)n_steps * kernels_per_step(g);
    return PHX_OK;
}

phx_status phx_step_adaptive(phx_grid* g, double t_end, const phx_adaptive* ctl) {
    if (!g || !ctl) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!g->has_params) return fail(g, PHX_ERR_BAD_STATE, "phx_step_adaptive: call phx_set_params first");
    if (g->d.integrator != PHX_INT_DP54) return fail(g, PHX_ERR_UNSUPPORTED, "phx_step_adaptive: create the grid with integrator = PHX_INT_DP54");
    if (g->d.noise) return fail(g, PHX_ERR_UNSUPPORTED, "phx_step_adaptive: not with noise (a Wiener increment cannot be re-drawn for a rejected step)");
    if (!(ctl->atol >= 0) || !(ctl->rtol >= 0) || !(ctl->atol + ctl->rtol > 0) || !(ctl->h_min > 0) || !(ctl->h_max >= ctl->h_min) ||
        !(ctl->h_init > 0) || !std::isfinite(t_end) || ctl->max_attempts < 0)
        return fail(g, PHX_ERR_INVALID_ARG, "phx_step_adaptive: bad tolerances or step-size bounds");
    // the integrator works on psi / n (and acc / nacc, ya / yb as scratch): bring the state home from the fused step's ping-pong
    { phx_status s = normalise_state(g); if (s) return s; }
    if (!g->gdp) {
        PHX_CUDA(g, g->d.prec == PHX_C64 ? build_dp_graph<double>(g) : build_dp_graph<float>(g));
    }
    // call parameters -> head of the device control block (t_end .. max_attempts are its first members)
    struct { double t_end, atol, rtol, h_init, h_min, h_max; long long max_attempts; } head = {
        t_end, ctl->atol, ctl->rtol, ctl->h_init, ctl->h_min, ctl->h_max, (long long)ctl->max_attempts};
    static_assert(offsetof(DpCtl, t) == sizeof(head), "DpCtl head layout");
    PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.dpctl, &head, sizeof(head), cudaMemcpyHostToDevice, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));   // (`head` is a stack variable: the staged copy must have left it)
    PHX_CUDA(g, cudaGraphLaunch(g->gdp, g->stream));
    g->launches += 1;                                 // (graph launches; the kernels inside are counted by phx_get_adaptive_state)
    return PHX_OK;
}

phx_status phx_get_adaptive_state(phx_grid* g, phx_adaptive_state* out, int32_t* log_accept, int32_t* log_q, double* log_h,
                                  double* log_err, int64_t log_cap, int64_t* n_log) {
    if (!g || !out) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (g->d.integrator != PHX_INT_DP54) return fail(g, PHX_ERR_UNSUPPORTED, "phx_get_adaptive_state: not an adaptive grid");
    DpCtl c;
    PHX_CUDA(g, cudaMemcpyAsync(&c, g->ws + g->L.dpctl, sizeof(c), cudaMemcpyDeviceToHost, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    out->t = c.t;
    out->h_next = c.h;
    out->n_accept = c.n_accept;
    out->n_reject = c.n_reject;
    out->attempts = c.attempts;
    out->err_last = c.err_last;
    int64_t n = c.log_count < DP_LOG_CAP ? c.log_count : DP_LOG_CAP;
    if (n > log_cap) n = log_cap;
    if (n < 0) n = 0;
    if (n_log) *n_log = n;
    if (n > 0) {
        if (log_accept) PHX_CUDA(g, cudaMemcpy(log_accept, c.log_accept, n * sizeof(int), cudaMemcpyDeviceToHost));
        if (log_q) PHX_CUDA(g, cudaMemcpy(log_q, c.log_q, n * sizeof(int), cudaMemcpyDeviceToHost));
        if (log_h) PHX_CUDA(g, cudaMemcpy(log_h, c.log_h, n * sizeof(double), cudaMemcpyDeviceToHost));
        if (log_err) PHX_CUDA(g, cudaMemcpy(log_err, c.log_err, n * sizeof(double), cudaMemcpyDeviceToHost));
    }
    return PHX_OK;
}

phx_status phx_set_time(phx_grid* g, double t, double h_next) {
    if (!g || !std::isfinite(t)) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (g->d.integrator != PHX_INT_DP54) return fail(g, PHX_ERR_UNSUPPORTED, "phx_set_time: not an adaptive grid");
    DpCtl c;
    PHX_CUDA(g, cudaMemcpyAsync(&c, g->ws + g->L.dpctl, sizeof(c), cudaMemcpyDeviceToHost, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    c.t = t;
    c.h = h_next > 0 ? h_next : 0.0;
    c.n_accept = c.n_reject = 0;
    c.k1_valid = 0;
    PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.dpctl, &c, sizeof(c), cudaMemcpyHostToDevice, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    return PHX_OK;
}

phx_status phx_get_step(const phx_grid* g, uint64_t* step) {
    if (!g || !step) return PHX_ERR_INVALID_ARG;
    *step = g->step_host;
    return PHX_OK;
}

phx_status phx_set_step(phx_grid* g, uint64_t step) {
    if (!g) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    const uint64_t slots[2] = {step, step};
    PHX_CUDA(g, cudaMemcpyAsync(g->ws + g->L.step, slots, sizeof(slots), cudaMemcpyHostToDevice, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    g->step_host = step;
    return PHX_OK;
}

phx_status phx_ensemble_mean_density(phx_grid* g, phx_field f, void* dst, phx_mem where) {
    if (!g || !dst || (where != PHX_HOST && where != PHX_DEVICE)) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (f != PHX_PSI && f != PHX_PSI_MINUS) return PHX_ERR_INVALID_ARG;
    if (!field_present(g, f)) return fail(g, PHX_ERR_UNSUPPORTED, "phx_ensemble_mean_density: field not present");
    size_t bytes;
    void* psi = field_ptr(g, f, &bytes);
    void* scratch = g->ws + g->L.yb[0];   // dead between steps in every variant
    PHX_CUDA(g, launch_ensemble_mean(psi, scratch, g->d.prec == PHX_C64, plane_cells(g), g->d.batch, g->stream));
    g->launches += 1;
    return copy_out(g, dst, scratch, plane_cells(g) * real_bytes(g), where);
}

phx_status phx_check_finite(phx_grid* g, int32_t* all_finite) {
    if (!g || !all_finite) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    int* flag = (int*)(g->ws + g->L.step + 64);          // (the counter slots take the first 16 of the 256 bytes)
    PHX_CUDA(g, cudaMemsetAsync(flag, 0, sizeof(int), g->stream));
    for (int f = PHX_PSI; f <= PHX_N_MINUS; ++f) {
        if (!field_present(g, f)) continue;
        size_t bytes;
        const void* p = field_ptr(g, f, &bytes);
        PHX_CUDA(g, launch_check_finite(p, bytes / real_bytes(g), g->d.prec == PHX_C64, flag, g->stream));
        g->launches += 1;
    }
    int host = 0;
    PHX_CUDA(g, cudaMemcpyAsync(&host, flag, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    *all_finite = host == 0;
    return PHX_OK;
}

phx_status phx_get_coeffs(const phx_grid* g, double* out, int32_t n) {
    if (!g || !out || n != PHX_NCOEF) return PHX_ERR_INVALID_ARG;
    if (!g->has_params) return PHX_ERR_BAD_STATE;
    std::memcpy(out, g->coef, sizeof(double) * PHX_NCOEF);
    return PHX_OK;
}

phx_status phx_debug_noise_u32(phx_grid* g, uint64_t step, uint32_t* dst, phx_mem where) {
    if (!g || !dst || (where != PHX_HOST && where != PHX_DEVICE)) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (!g->has_params) return fail(g, PHX_ERR_BAD_STATE, "phx_debug_noise_u32: call phx_set_params first (seed)");
    const size_t plane = plane_cells(g);
    if (where == PHX_DEVICE) {
        PHX_CUDA(g, launch_noise_words(dst, g->prm.seed, step, plane, 0, g->d.batch, g->stream));
        PHX_CUDA(g, cudaStreamSynchronize(g->stream));
        return PHX_OK;
    }
    // stage through the buffers that are dead between steps (yb, acc), one chunk of realisations at a time
    const size_t per_real = plane * 16;
    const size_t chunk = g->L.scratch_bytes / per_real;
    if (chunk < 1) return fail(g, PHX_ERR_UNSUPPORTED, "phx_debug_noise_u32: scratch too small");
    uint32_t* scratch = (uint32_t*)(g->ws + g->L.yb[0]);
    for (size_t r0 = 0; r0 < (size_t)g->d.batch; r0 += chunk) {
        const size_t nr = (size_t)g->d.batch - r0 < chunk ? (size_t)g->d.batch - r0 : chunk;
        PHX_CUDA(g, launch_noise_words(scratch, g->prm.seed, step, plane, (int)r0, (int)nr, g->stream));
        phx_status s = copy_out(g, dst + r0 * plane * 4, scratch, nr * per_real, PHX_HOST);
        if (s) return s;
    }
    return PHX_OK;
}

phx_status phx_select_variant(phx_grid* g, int32_t variant) {
    if (!g) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    if (variant != PHX_VARIANT_AUTO && variant != PHX_VARIANT_STAGE && !(variant == PHX_VARIANT_STEP && step_variant_ok(g)) &&
        !(variant == PHX_VARIANT_RESIDENT && resident_variant_ok(g)))
        return fail(g, PHX_ERR_UNSUPPORTED, "phx_select_variant: variant not available for this grid/model");
    g->variant_req = variant;
    return apply_variant(g);
}

phx_status phx_get_variant(const phx_grid* g, int32_t* variant) {
    if (!g || !variant) return PHX_ERR_INVALID_ARG;
    *variant = g->variant;
    return PHX_OK;
}

phx_status phx_get_launch_count(const phx_grid* g, uint64_t* launches) {
    if (!g || !launches) return PHX_ERR_INVALID_ARG;
    *launches = g->launches;
    return PHX_OK;
}

phx_status phx_set_tuning(phx_grid* g, const char* key, int32_t value) {
    if (!g || !key) return PHX_ERR_INVALID_ARG;
    if (!std::strcmp(key, "rows")) {
        if (value < 1 || value > 4096) return PHX_ERR_INVALID_ARG;
        g->rows = value;
    } else if (!std::strcmp(key, "vec")) {
        if (value != 1 && value != 2) return PHX_ERR_INVALID_ARG;
        if (value == 2 && g->d.nx % 2 != 0) return fail(g, PHX_ERR_UNSUPPORTED, "vec=2 needs even nx");
        g->vec = value;
    } else if (!std::strcmp(key, "step_ly")) {        // variant STEP: rows per chunk (0 = automatic)
        if (value < 0 || value > (1 << 20)) return PHX_ERR_INVALID_ARG;
        g->step_ly = value;
    } else if (!std::strcmp(key, "step_vec")) {       // variant STEP: cells per lane (0 = automatic)
        if (value != 0 && value != 1 && value != 2 && value != 4) return PHX_ERR_INVALID_ARG;
        if (value >= 2 && g->d.nx % value != 0) return fail(g, PHX_ERR_UNSUPPORTED, "step_vec>1 needs nx a multiple of it");
        if (value == 4 && (g->d.model != PHX_SCALAR || g->d.prec != PHX_C32)) return fail(g, PHX_ERR_UNSUPPORTED, "step_vec=4 exists for the scalar fp32 model only");
        if (value == 2 && g->d.prec == PHX_C64 && g->d.model != PHX_SCALAR) return fail(g, PHX_ERR_UNSUPPORTED, "step_vec=2 in fp64 exists for the scalar model only");
        g->step_vec = value;
    } else if (!std::strcmp(key, "step_warps")) {     // variant STEP: warps per CTA (0 = automatic)
        if (value < 0 || value > PHX_STEP_WARPS) return PHX_ERR_INVALID_ARG;
        g->step_warps = value;
    } else if (!std::strcmp(key, "step_bulk")) {      // variant STEP fetch path: -1 automatic, 0 register loads, 1 shared-memory ring (cp.async / TMA)
        if (value < -1 || value > 1) return PHX_ERR_INVALID_ARG;
        g->step_bulk = value;
    } else if (!std::strcmp(key, "step_xch")) {       // variant STEP exchanging strips: -1 automatic (wherever the row fits), 0 off
        if (value < -1 || value > 1) return PHX_ERR_INVALID_ARG;
        g->step_xch = value;
    } else if (!std::strcmp(key, "resident_cluster")) {   // variant RESIDENT on a thread-block cluster: -1 automatic, 0 never, 1 whenever it applies
        if (value < -1 || value > 1) return PHX_ERR_INVALID_ARG;
        g->resident_cluster = value;
        resolve_variant(g);
    } else if (!std::strcmp(key, "step_pdl")) {       // variant STEP programmatic dependent launches inside a graph: -1 automatic, 0 off, 1 on
        if (value < -1 || value > 1) return PHX_ERR_INVALID_ARG;
        g->step_pdl = value;
    } else if (!std::strcmp(key, "step_side")) {      // variant STEP side launch for a ragged last strip: 1 on; -1 (automatic) and 0: off
        if (value < -1 || value > 1) return PHX_ERR_INVALID_ARG;
        g->step_side = value;
    } else if (!std::strcmp(key, "async_host_copies")) {   // 1: phx_set_field / phx_read_field with PHX_HOST do not synchronise
        if (value != 0 && value != 1) return PHX_ERR_INVALID_ARG;
        g->async_host = value;
        return PHX_OK;                                 // (no effect on the launch plan: keep the captured graphs)
    } else if (!std::strcmp(key, "graph_steps")) {
        if (value < 1 || value > 256) return PHX_ERR_INVALID_ARG;
        g->graph_steps = value;
    } else {
        return fail(g, PHX_ERR_UNSUPPORTED, "phx_set_tuning: unknown key");
    }
    drop_graphs(g);
    return PHX_OK;
}

phx_status phx_sync(phx_grid* g) {
    if (!g) return PHX_ERR_INVALID_ARG;
    if (g->sticky != cudaSuccess) return PHX_ERR_CUDA;
    PHX_CUDA(g, cudaStreamSynchronize(g->stream));
    return PHX_OK;
}

const char* phx_last_error(const phx_grid* g) { return g ? g->err.c_str() : "null handle"; }

void phx_destroy_grid(phx_grid* g) {
    if (!g) return;
    drop_graphs(g);
    if (g->cap_stream) cudaStreamDestroy(g->cap_stream);
    if (g->side_stream) cudaStreamDestroy(g->side_stream);
    if (g->ev_fork) cudaEventDestroy(g->ev_fork);
    if (g->ev_join) cudaEventDestroy(g->ev_join);
    delete g;
}

}  // extern "C"
