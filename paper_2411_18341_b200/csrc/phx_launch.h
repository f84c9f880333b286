// phx_launch.h -- host-side entry points of the kernel translation units (internal to libphx).
#pragma once

#include "phx_common.cuh"

// Most warps per CTA of variant STEP (the warps of a CTA are independent: adjacent strips, no barrier between them; the
// launch plan takes 1 or PHX_STEP_WARPS per CTA, whichever leaves fewer warp slots idle: StepArgs::wpc).
#ifndef PHX_STEP_WARPS
#define PHX_STEP_WARPS 2
#endif

// Variant STEP, exchanging strips (phx_step.cuh, XCH): most warps per CTA; the warps of a CTA tile the whole row.
#ifndef PHX_STEP_XWARPS
#define PHX_STEP_XWARPS 8
#endif
// How the warps of a row wait for each other: 0 = a progress counter per warp, polled (neighbours drift by up to one iteration);
// 1 = one named barrier per iteration (lockstep, no branch in the row loop).
// (measured on cfg5, 512 x 256^2 reservoir + noise: barrier 99.9, counters 74.6, no exchange 88.5 Gcell*step/s: the spin loop
// splits every phase of the row loop into basic blocks)
#ifndef PHX_XCH_SYNC
#define PHX_XCH_SYNC 1
#endif

// Variant STEP: row iterations a fetch leads its first use by, and the ring length / unroll factor of the row loop.
// (LEAD = 2 costs registers and is slower everywhere: 200.6 against 207.5 Gcell*step/s at 4096^2 fp32, spills in the spinor.)
#ifndef PHX_STEP_LEAD
#define PHX_STEP_LEAD 1
#endif
#define PHX_STEP_RING (4 + PHX_STEP_LEAD)
// The exchanging strips fetch two rows ahead: a warp that waits for a load holds the whole row's barrier up, and the kernels
// have the registers (cfg5: 105.0 against 102.2 Gcell*step/s).
#ifndef PHX_STEP_XLEAD
#define PHX_STEP_XLEAD 2
#endif
// Leave the unrolled row loop in the middle of its last pass (a chunk of ly rows costs ly + 6 iterations instead of the next
// multiple of the ring length).  The exit test splits the loop body into one basic block per phase, which costs the other
// kernels more than the saved iterations give back (same-run A/B: 4096^2 scalar fp32 4 cells per lane 213 against 205
// Gcell*step/s and 1024^2 scalar fp64 2 cells per lane 70.8 against 64.3 with the exit; cfg3 reservoir 141.6 against 147.6,
// 1024^2 fp32 101.8 against 110.3, a single 64^2 fp64 grid 5.4 against 3.8 us per step without): taken by those two only.
#ifndef PHX_STEP_EARLY_EXIT
#define PHX_STEP_EARLY_EXIT 1
#endif
namespace phx {
constexpr bool step_early_exit(bool prec64, int model, int vec) {
    return PHX_STEP_EARLY_EXIT && model == 0 && ((!prec64 && vec == 4) || (prec64 && vec == 2));
}
}
// Bulk-copy fetch path of variant STEP: stages of the per-warp shared-memory ring (rows in flight = DEPTH - 1); power of 2.
#ifndef PHX_STEP_DEPTH
#define PHX_STEP_DEPTH 8
#endif
namespace phx {
// Which flavour of the shared-memory ring a (precision, model) pair gets, and how deep.  cp.async (every lane copies its own
// cells, no mbarrier): measured FASTER than the register loads on the reservoir model in complex fp32 (five arrays per row;
// cfg3 4096^2: 155-160 against 144-147 Gcell*step/s at depth 8; cfg5-shaped ensembles without exchanging strips 98.6 against
// 88.7) and marginally on the scalar model in complex fp64 (102.2-105.5 against 100.7-102.9 at depth 4): those two take it
// by default from 512^2 cells up (step_ring_auto; phx_api.cu: step_bulk).  Everything else keeps the TMA bulk-copy flavour as an opt-in
// (slower than the register loads everywhere: profiles/r02_tma_vs_register_fetch.md).
// (vec = cells per lane.)  The scalar fp32 kernel with 2 or 1 cells per lane gains 2-3 % as well (1024^2 116.2 against 113.4,
// 1536^2 163.8 against 158.6); with 4 cells per lane it loses 11 % and keeps register loads (its ring, the TMA flavour, is opt-in).
#ifndef PHX_RING_CPA_V4
#define PHX_RING_CPA_V4 0
#endif
constexpr bool step_ring_cpasync(bool prec64, int model, int vec) {
    return (!prec64 && model == 1) || (prec64 && model == 0) || (!prec64 && model == 0 && (vec <= 2 || PHX_RING_CPA_V4));
}
constexpr int step_ring_depth(bool prec64, int model) { return (prec64 && model == 0) ? 4 : PHX_STEP_DEPTH; }
constexpr bool step_ring_auto(bool prec64, int model, int vec) { return step_ring_cpasync(prec64, model, vec) && (vec == 2 || (prec64 && vec == 1)); }
// The exchanging strips of the reservoir model in complex fp32 (cfg5) fetch through the cp.async ring (106.5 against 101.6
// Gcell*step/s) and then need only one row of register lead (109.6 against 106.5 with two).
#ifndef PHX_XCH_RING
#define PHX_XCH_RING 1
#endif
constexpr bool step_xch_ringed(bool prec64, int model, int vec) { return PHX_XCH_RING && !prec64 && model == 1 && vec == 2; }
constexpr int step_xch_lead(bool prec64, int model, int vec) { return step_xch_ringed(prec64, model, vec) ? 1 : PHX_STEP_XLEAD; }
}

namespace phx {

template <typename T> struct StageArgs;

#define PHX_DECL_STAGE(P, T)                                                                                              \
    cudaError_t launch_stage_##P##_0(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_1(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_2(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t); \
    cudaError_t launch_stage_##P##_3(const StageArgs<T>&, int stage, bool noise, int vec, dim3 grid, dim3 block, cudaStream_t);
PHX_DECL_STAGE(32, float)
PHX_DECL_STAGE(64, double)
#undef PHX_DECL_STAGE

template <typename T> struct StepArgs;

#define PHX_DECL_STEP(P, T)                                                                                      \
    cudaError_t launch_step_##P##_0(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_1(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_2(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_step_##P##_3(const StepArgs<T>&, bool noise, bool zbc, bool iso, bool bulk, int vec, dim3 grid, cudaStream_t); \
    int occupancy_step_##P##_0(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_1(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_2(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);                                          \
    int occupancy_step_##P##_3(bool noise, bool zbc, bool iso, bool drive, bool bulk, int vec);
PHX_DECL_STEP(32, float)
PHX_DECL_STEP(64, double)
#undef PHX_DECL_STEP

// phx_stepx_inst.cu: the fused step with exchanging strips (scalar and reservoir models, periodic, no drive).  `vec` must be
// one the precision and model have (stepx_has_vec); the CTA has a.wpc warps; occupancy = resident CTAs of `warps` warps per SM.
#define PHX_DECL_STEPX(P, T)                                                                                  \
    cudaError_t launch_stepx_##P##_0(const StepArgs<T>&, bool noise, bool iso, int vec, dim3 grid, cudaStream_t); \
    cudaError_t launch_stepx_##P##_1(const StepArgs<T>&, bool noise, bool iso, int vec, dim3 grid, cudaStream_t); \
    int occupancy_stepx_##P##_0(bool noise, bool iso, int vec, int warps);                                        \
    int occupancy_stepx_##P##_1(bool noise, bool iso, int vec, int warps);
PHX_DECL_STEPX(32, float)
PHX_DECL_STEPX(64, double)
#undef PHX_DECL_STEPX
// cells per lane the exchanging strips are instantiated with: complex fp32 2 (scalar also 4), complex fp64 1 (scalar also 2)
inline bool stepx_has_vec(int prec64, int model, int vec) {
    if (model > 1) return false;
    if (!prec64) return vec == 2 || (vec == 4 && model == 0);
    return vec == 1 || (vec == 2 && model == 0);
}

// phx_resident.cu: variant RESIDENT (a small grid on chip for all steps of one launch)
#ifndef PHX_RESIDENT_THREADS
#define PHX_RESIDENT_THREADS 512
#endif
template <typename T>
struct ResidentArgs {
    Geom geo;
    Coef<T> k;
    typename Cx<T>::type* psi;      // state [batch][ny][nx], advanced in place
    T* n;                           // reservoir state, or nullptr
    const T* V;                     // [ny][nx] or nullptr
    const T* P;                     // [ny][nx] or nullptr
    uint64_t* step_slots;           // both device step-counter slots receive step0 + n_steps
    uint64_t step0;                 // completed steps before this launch
    int n_steps;
    uint32_t seed;
    const typename Cx<T>::type* E;  // drive amplitude [ny][nx] or nullptr (cluster form of the scalar model only)
};
int resident_cpt(size_t cells, int prec64, bool res);     // cells per thread, 0 = the grid does not fit
cudaError_t launch_resident_32(const ResidentArgs<float>&, bool res, bool noise, cudaStream_t);
cudaError_t launch_resident_64(const ResidentArgs<double>&, bool res, bool noise, cudaStream_t);
// cluster form: one realisation on a thread-block cluster of 2-8 CTAs (row slabs, halo rows through distributed shared memory)
int resident_cluster_size(int nx, int ny, int prec64, bool res);   // 0 = does not apply
bool resident_drive_ok(int nx, int ny, int prec64);                // a driven scalar grid fits the cluster form
cudaError_t launch_resident_cluster_32(const ResidentArgs<float>&, bool res, bool noise, cudaStream_t);
cudaError_t launch_resident_cluster_64(const ResidentArgs<double>&, bool res, bool noise, cudaStream_t);

// phx_aux.cu: small helper kernels
cudaError_t launch_check_finite(const void* data, size_t n_reals, int prec64, int* flag, cudaStream_t);   // *flag <- 1 on NaN / Inf
cudaError_t launch_ensemble_mean(const void* psi, void* out, int prec64, size_t plane, int batch, cudaStream_t);
cudaError_t launch_noise_words(uint32_t* out, uint32_t seed, uint64_t step, size_t plane, int r0, int batch, cudaStream_t);

}  // namespace phx
